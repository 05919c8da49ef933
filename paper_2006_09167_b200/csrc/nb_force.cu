// nb_force.cu -- (a7) the cluster-pair force kernel and (a8) force reduction / outputs.
//
// interactions between i-clusters and a joint list of j-clusters, skipped
// per cluster pair through the interaction mask; Newton's third law so both i and j forces are
// reduced (L133); exclusions as bitmasks applied together with the cut-off (L135); analytical
// Ewald correction on FMA hardware (L137); one kernel per combination of electrostatics and
// energy/no-energy to avoid conditionals (L139).
//
// Thread mapping (differs from the paper's 8x4-per-warp tiles): one thread
// block = one warp = one i-cluster working through one segment of the compact inner list that the
// prune kernel wrote for it.  The 8 i atoms sit in registers of every lane as 4 packed pairs.
// Lanes own j atoms: an unmasked step takes the next 32 listed j atoms (the inner list is kept per j atom),
// a masked step 4 whole j-clusters with their exclusion masks; every lane evaluates its j atom
// against the 8 i atoms, two at a time with packed FP32x2 instructions.  Consequences: no shuffle
// in the inner loop (the j force is private to its lane and leaves with ONE vector atomic per j
// atom per step, i.e. atomics at cluster granularity), no per-pair shared-memory load of i data,
// no mask tests (the list holds survivors only), and the i forces (8 x 3 registers) are reduced
// across lanes once per segment.
#include "nb_internal.h"

#include <algorithm>
#include <mutex>

#include "ewald_corr_coeffs.h"

namespace {

struct ForceArgs {
    const int4* units;          // work units {entry slot, batch begin, batch end, sci}, canonical order (k_count_pairs)
    const int2* jl;
    const uint32_t* plane;
    const float4* xq;
    const int* type_slot;
    const float4* ljrow;        // paired LJ rows per i-cluster (k_ljrows)
    const unsigned long long* masks;
    const int4* segd;           // compact inner list, see nb_internal.h
    const int2* seg_cnt[2];
    const int* il[2];
    const int2* ilm[2];
    unsigned bufmask;           // which inner buffer each rolling part lives in (nb_prune_overlapped), 0 = all in buffer 0
    const int32_t* seg_part;    // rolling part of every segment under buf_nparts (read only while bufmask != 0)
    int nparts, nunits;
    // the fused first prune (k_force<..., PRUNE = true>): outer list in, inner list (buffer 0) out
    const int2* ol_cnt;
    const int* olu;
    const int2* olm;
    int32_t* il_w;
    int2* ilm_w;
    int2* seg_cnt_w;
    float rl2;                  // fl32(rlist_inner^2), reading A12
    int cj_dummy;
    cudaStream_t launch_stream;   // nullptr: the context's stream
    int seg_base, seg_count;    // launch over the segments [seg_base, seg_base + seg_count) of the force order (count 0: all
                                // of them): the local / non-local kernels of nb_forces_local / nb_forces_nonlocal
    float4* f4;
    double* fshift;     // [27*3]
    double* energies;   // [2]
    NbConst kc;
};

__device__ __forceinline__ void red_add_v4(float4* addr, float x, float y, float z)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(x), "f"(y), "f"(z), "f"(0.0f)
                 : "memory");
}

// Single-instruction MUFU forms: the arguments are clamped away from zero/denormals by the
// caller (r^2 >= 1e-6 or distinct atoms, monic Q(r^2) >= 1/30), so the denormal fix-up code of rsqrtf()/__fdividef() is dead weight.
__device__ __forceinline__ float rsqrt_fast(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_fast(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Packed FP32x2 arithmetic (sm_100 FFMA2/FMUL2/FADD2): one issue slot per two pair evaluations.
// The FP32 pipe rate in flop/s is the same as for scalar FFMA (measured), but the kernel is
// issue-bound in scalar form, so halving the issue slots of the
// FP32-pipe work is what moves it towards the FP32 roofline.
__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }

// beta^3 h(z) for two pairs, as P4(r^2)/Q5(r^2) with beta folded into the coefficients and Q made
// monic (P divided by Q's leading coefficient): Q's first Horner step is then an FADD2 with one
// constant operand, and P's first step takes its addend from a register pair (p3) kept by the
// caller -- an FFMA2 cannot take two constant-bank operands, ptxas would rebuild them with MOVs.
__device__ __forceinline__ float2 ewald_bh2(float2 r2, const NbConst& K, const float2 p3)
{
    float2 p = fma2(K.ewp2[4], r2, p3);
    float2 q = add2(r2, K.ewq2[4]);
    q = fma2(q, r2, K.ewq2[3]);
    p = fma2(p, r2, K.ewp2[2]);
    q = fma2(q, r2, K.ewq2[2]);
    p = fma2(p, r2, K.ewp2[1]);
    q = fma2(q, r2, K.ewq2[1]);
    p = fma2(p, r2, K.ewp2[0]);
    q = fma2(q, r2, K.ewq2[0]);
    return mul2(p, f2(rcp_fast(q.x), rcp_fast(q.y)));
}

// The 8 i atoms of the warp's cluster as 4 packed pairs (atoms 2p, 2p+1); charges carry epsfac.
struct IAtoms {
    float2 x[4], y[4], z[4], q[4];
};

// One step: this lane's j atom (xj; ljj points at the lane's j-type column of the warp's paired LJ
// table, stride `ljs` float4 between i-atom pairs) against the 8 i atoms, two at a time.
// MASKED: cbyte/mbyte carry the lane's 8 "counted"/"interacts" bits (reading A4: an excluded pair
// keeps the Ewald/RF correction, loses LJ and the 1/r part).
// TWIN: twin cut-offs, LJ only below rc_vdw <= rc.
// PRUNE: the fused first prune; returns whether some counted pair of this lane's j atom is
// within rlist_inner, decided on the same r^2 (the exact A12 arithmetic: I holds fmaf(s, L, x_a), and
// x_a' + (-x_b) = x_a' - x_b, fma2(dz,dz, fma2(dy,dy, dx*dx)) round like the oracle's scalar forms).
// Returns the NEGATED j force in (fjx, fjy, fjz) pairs (sum the halves and negate).
template <int COUL, bool ENERGY, bool MASKED, bool TWIN, bool PRUNE>
__device__ __forceinline__ bool pair_step(const NbConst& K, const float4* __restrict__ ljj, const int ljs, const IAtoms& I,
                                          float2 (&fix)[4], float2 (&fiy)[4], float2 (&fiz)[4], float& elj, float& ecoul,
                                          const float4 xj, unsigned cbyte, unsigned mbyte, float2& fjx, float2& fjy,
                                          float2& fjz, const float2 p3, const float rl2)
{
    const float2 nxj = f2(-xj.x), nyj = f2(-xj.y), nzj = f2(-xj.z), qj = f2(xj.w);
    fjx = f2(0.f); fjy = f2(0.f); fjz = f2(0.f);
    bool found = false;
#pragma unroll
    for (int p = 0; p < 4; p++) {
        const float2 dx = add2(I.x[p], nxj), dy = add2(I.y[p], nyj), dz = add2(I.z[p], nzj);
        const float2 r2u = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
        if (PRUNE) {
            if (MASKED) found = found || (r2u.x < rl2 && ((cbyte >> (2 * p)) & 1u)) || (r2u.y < rl2 && ((cbyte >> (2 * p + 1)) & 1u));
            else found = found || r2u.x < rl2 || r2u.y < rl2;
        }
        // A7: interact iff r^2 < rc^2 (strict), applied with compare + select on the ALU pipe, which
        // has slack (the FP32 pipe is the bound; a saturating-FMA 0/1 factor there was measured 1 %
        // slower).  MASKED steps also clamp r^2 so that self pairs stay finite; unmasked steps have no
        // r = 0 pairs (padding atoms sit at distinct finite positions, nb_grid.cu).
        bool w0 = true, w1 = true;
        float2 r2 = r2u;
        if (MASKED) {
            w0 = r2u.x < K.rc2 && ((cbyte >> (2 * p)) & 1u);
            w1 = r2u.y < K.rc2 && ((cbyte >> (2 * p + 1)) & 1u);
            r2 = f2(fmaxf(r2u.x, 1e-6f), fmaxf(r2u.y, 1e-6f));
        } else {
            w0 = r2u.x < K.rc2;
            w1 = r2u.y < K.rc2;
        }
        const float2 rinv = f2(rsqrt_fast(r2.x), rsqrt_fast(r2.y));
        const float2 rinv2 = mul2(rinv, rinv);
        const float4 c = ljj[p * ljs];                        // (-6 c6_a, -6 c6_b, 12 c12_a, 12 c12_b)
        const float2 nc6 = f2(c.x, c.y), c12 = f2(c.z, c.w);
        const float2 rinv6 = mul2(mul2(rinv2, rinv2), rinv2);
        float2 flj = mul2(fma2(c12, rinv6, nc6), rinv6);
        const bool v0 = !TWIN || r2u.x < K.rcv2, v1 = !TWIN || r2u.y < K.rcv2;   // LJ cut-off (twin cut-offs)
        if (TWIN) flj = f2(v0 ? flj.x : 0.f, v1 ? flj.y : 0.f);
        const float2 qq = mul2(I.q[p], qj);                   // epsfac folded into the i charge
        float2 t1 = COUL == NB_COUL_NONE ? flj : fma2(qq, rinv, flj);   // (F_lj + A/r) r
        float2 mf = f2(1.f);
        if (MASKED) {
            mf = f2(((mbyte >> (2 * p)) & 1u) ? 1.f : 0.f, ((mbyte >> (2 * p + 1)) & 1u) ? 1.f : 0.f);
            t1 = mul2(t1, mf);                                // excluded pair: only the correction term
        }
        float2 fs, bh = f2(0.f);
        if (COUL == NB_COUL_EWALD) {
            bh = ewald_bh2(r2, K, p3);
            fs = fma2(rinv2, t1, neg2(mul2(qq, bh)));         // F/r = (F_lj r + A m/r)/r^2 - A beta^3 h
        } else if (COUL == NB_COUL_RF) {
            fs = fma2(rinv2, t1, neg2(mul2(qq, f2(K.two_krf))));   // F/r = ... - 2 A k_rf
        } else {
            fs = mul2(rinv2, t1);                             // LJ only: charges are ignored
        }
        fs = f2(w0 ? fs.x : 0.f, w1 ? fs.y : 0.f);
        fix[p] = fma2(fs, dx, fix[p]);
        fiy[p] = fma2(fs, dy, fiy[p]);
        fiz[p] = fma2(fs, dz, fiz[p]);
        fjx = fma2(fs, dx, fjx);
        fjy = fma2(fs, dy, fjy);
        fjz = fma2(fs, dz, fjz);
        if (ENERGY) {
            // V_lj = c12 (r^-12 - rc^-12) - c6 (r^-6 - rc^-6), table holds (-6 c6, 12 c12)
            const float2 a12 = fma2(rinv6, rinv6, f2(-K.lj_sh12)), a6 = add2(rinv6, f2(-K.lj_sh6));
            const float2 vlj = fma2(mul2(c12, f2(1.f / 12.f)), a12, mul2(mul2(nc6, f2(1.f / 6.f)), a6));
            float2 vc;
            if (COUL == NB_COUL_EWALD) {
                // beta e(z) = r^2 beta^3 h(z) + beta (2/sqrt(pi)) exp(-z)
                const float2 ex = f2(__expf(-K.beta2 * r2.x), __expf(-K.beta2 * r2.y));
                const float2 be = fma2(r2, bh, mul2(f2(K.beta * 1.1283791671f), ex));
                vc = mul2(qq, add2(mul2(mf, add2(rinv, f2(-K.ewald_shift))), neg2(be)));
            } else if (COUL == NB_COUL_RF) {
                vc = mul2(qq, fma2(mf, rinv, fma2(f2(K.krf), r2, f2(-K.crf))));
            } else {
                vc = f2(0.f);
            }
            const float2 vl = mul2(mf, vlj);
            elj += (w0 && v0 ? vl.x : 0.f) + (w1 && v1 ? vl.y : 0.f);
            ecoul += (w0 ? vc.x : 0.f) + (w1 ? vc.y : 0.f);
        }
    }
    return found;
}

// PRUNE = false: the inner list (listed j atoms, 32 per step; masked cluster pairs, 4 per step).
// PRUNE = true: the fused first prune of a freshly searched list: the same kernel walks
// the OUTER list (whole j-clusters, 4 per step), evaluates the forces, and writes the inner list from
// the r^2 values it has anyway -- one ballot per step, as in nb_prune.cu's kernel.
template <int COUL, bool ENERGY, bool TWIN, bool PRUNE>
__global__ void __launch_bounds__(32, PRUNE ? 8 : 16) k_force(ForceArgs A)
{
    // Paired LJ table of this block's i-cluster: s_ljp[p*nt1 + tj] = (-6c6, -6c6', 12c12, 12c12') of the
    // i atoms 2p, 2p+1 against j type tj: one LDS.128 feeds both packed operands.
    extern __shared__ float4 s_ljp[];
    nb_pdl_wait();
    nb_pdl_trigger();
    const NbConst& K = A.kc;
    const int lane = threadIdx.x & 31, g = lane >> 3, k = lane & 7;
    const int seg = blockIdx.x + A.seg_base;
    const int4 sd = A.segd[seg];
    // (the part comes from a table written when nparts changes: deriving it from the unit index costs a 64-bit division)
    const int buf = PRUNE || !A.bufmask ? 0 : (int)((A.bufmask >> A.seg_part[seg]) & 1u);
    // PRUNE: outer counts {cluster pairs without a mask, with a mask}; else inner {j-atom entries, masked pairs}
    const int2 cnt = PRUNE ? A.ol_cnt[seg] : A.seg_cnt[buf][seg];
    const int ci = sd.z & 0x3ffffff, sid = sd.z >> 26, warp = ci & 7;
    const int nt1 = K.ntypes1;
    float4* ljw = s_ljp;
    // the rows were paired at search time (types do not change between searches): one coalesced load
    for (int i = lane; i < 4 * nt1; i += 32) ljw[i] = A.ljrow[(size_t)ci * 4 * nt1 + i];
    const int* __restrict__ il = (PRUNE ? A.olu : A.il[buf]) + sd.x;
    const int2* __restrict__ ilm = (PRUNE ? A.olm : A.ilm[buf]) + sd.y;
    int32_t* il_w = PRUNE ? A.il_w + sd.x : nullptr;
    int2* ilm_w = PRUNE ? A.ilm_w + sd.y : nullptr;
    int nu_w = 0, nm_w = 0;
    // unmasked steps: 32 listed j atoms per step, one per lane; PRUNE: the outer list, 4 whole clusters per step
    const int ns = PRUNE ? (cnt.x + 3) >> 2 : cnt.x >> 5;
    // this lane's j SLOT in step s.  PRUNE: the last step may be partly filled; its spare lanes take a dummy cluster
    // (far from everything: no force, no survivor; nb_grid.cu)
    auto entry = [&](int s) {
        if (!PRUNE) return il[32 * s + lane];
        const int idx = 4 * s + g, v = il[min(idx, max(cnt.x - 1, 0))];
        return (idx < cnt.x ? v : A.cj_dummy) * 8 + k;
    };
    // first list entries of both loops are requested before anything else is waited for
    int cj = 0, cj_n = 0;
    if (ns > 0) {
        cj = entry(0);                         // unmasked path: cj* hold this lane's j SLOT
        cj_n = entry(min(1, ns - 1));
    }
    // ... and so is the first step of the masked loop (its loads chain entry -> atoms -> mask)
    int2 ce_next = g < cnt.y ? ilm[g] : make_int2(ci, 0);
    int sx, sy, sz;
    nb_shift_vec(sid, sx, sy, sz);
    IAtoms I;
#pragma unroll
    for (int p = 0; p < 4; p++) {
        const float4 v0 = A.xq[ci * 8 + 2 * p], v1 = A.xq[ci * 8 + 2 * p + 1];
        I.x[p] = f2(fmaf((float)sx, K.box[0], v0.x), fmaf((float)sx, K.box[0], v1.x));
        I.y[p] = f2(fmaf((float)sy, K.box[1], v0.y), fmaf((float)sy, K.box[1], v1.y));
        I.z[p] = f2(fmaf((float)sz, K.box[2], v0.z), fmaf((float)sz, K.box[2], v1.z));
        I.q[p] = f2(K.epsfac * v0.w, K.epsfac * v1.w);
    }
    float2 fix[4], fiy[4], fiz[4];
#pragma unroll
    for (int p = 0; p < 4; p++) { fix[p] = f2(0.f); fiy[p] = f2(0.f); fiz[p] = f2(0.f); }
    float elj = 0.f, ecoul = 0.f;
    const float2 p3 = K.ewp2[3];
    float4 xj = make_float4(0.f, 0.f, 0.f, 0.f);
    int tj = 0;
    if (ns > 0) {   // j data of the first unmasked step: in flight during the masked steps
        xj = A.xq[cj];
        tj = A.type_slot[cj];
    }
    __syncwarp();

    // Cluster pairs with exclusion / self / diagonal masks.  (Software-pipelining this loop like the
    // unmasked one was measured slower.)
    for (int s = 0; s < cnt.y; s += 4) {
        const bool valid = s + g < cnt.y;
        const int2 ce = ce_next;
        if (s + 4 < cnt.y) ce_next = s + 4 + g < cnt.y ? ilm[s + 4 + g] : make_int2(ci, 0);
        const float4 xm = A.xq[ce.x * 8 + k];
        const int tm = A.type_slot[ce.x * 8 + k];
        const ulonglong2 mm = *reinterpret_cast<const ulonglong2*>(&A.masks[((size_t)ce.y * 8 + warp) * 2]);
        const unsigned cbyte = valid ? (unsigned)(mm.y >> (8 * k)) & 0xffu : 0u;
        const unsigned mbyte = (unsigned)(mm.x >> (8 * k)) & cbyte;
        float2 fjx, fjy, fjz;
        const bool found = pair_step<COUL, ENERGY, true, TWIN, PRUNE>(K, ljw + tm, nt1, I, fix, fiy, fiz, elj, ecoul, xm, cbyte,
                                                                      mbyte, fjx, fjy, fjz, p3, A.rl2);
        if (valid) red_add_v4(&A.f4[ce.x * 8 + k], -(fjx.x + fjx.y), -(fjy.x + fjy.y), -(fjz.x + fjz.y));
        if (PRUNE) {   // surviving cluster pairs of the step keep their {cj, mask ref}
            const unsigned gm = __ballot_sync(0xffffffffu, found);
            unsigned cm = gm | (gm >> 1);
            cm |= cm >> 2;
            cm = (cm | (cm >> 4)) & 0x01010101u;
            if ((cm >> lane) & 1u) ilm_w[nm_w + __popc(cm & ((1u << lane) - 1u))] = ce;
            nm_w += __popc(cm);
        }
    }

    // Cluster pairs without a mask: always full steps of 32 listed j atoms (PRUNE: 4 clusters, the last step
    // possibly partly filled).  ptxas schedules memory operations whose consumer is an iteration away at the
    // END of a step, so the j data is requested TWO steps ahead into registers (xj: this step, xj1: next
    // step, x2: the one after) and the list entries four steps ahead, indices clamped to the segment.
    int cj2 = 0, cj3 = 0;
    float4 xj1 = xj;
    int tj1 = tj;
    if (ns > 0) {
        cj2 = entry(min(2, ns - 1));
        cj3 = entry(min(3, ns - 1));
        xj1 = A.xq[cj_n];
        tj1 = A.type_slot[cj_n];
    }
    // Unrolled by the period of the register rotation below (3: no copies at the end of the body) in the force-only
    // flavour: 70.4 -> 68.3 us on config 2, 697 -> 673 us on config 3 with the j-atom list (it was slower with the
    // half-cluster list); the energy flavour, with more live registers, is faster unrolled by 2.  A prefetch distance of
    // three steps for the j data (unrolled by 4) measured the same as two.
#pragma unroll(ENERGY ? 2 : 3)
    for (int s = 0; s < ns; s++) {
        const int cj4 = entry(min(s + 4, ns - 1));
        const float4 x2 = A.xq[cj2];
        const int t2 = A.type_slot[cj2];
        float2 fjx, fjy, fjz;
        const bool found = pair_step<COUL, ENERGY, false, TWIN, PRUNE>(K, ljw + tj, nt1, I, fix, fiy, fiz, elj, ecoul, xj, 0xffu,
                                                                       0xffu, fjx, fjy, fjz, p3, A.rl2);
        red_add_v4(&A.f4[cj], -(fjx.x + fjx.y), -(fjy.x + fjy.y), -(fjz.x + fjz.y));
        if (PRUNE) {   // the j atoms of the step that have a partner within rlist_inner keep their slot
            const unsigned gm = __ballot_sync(0xffffffffu, found);
            if (found) il_w[nu_w + __popc(gm & ((1u << lane) - 1u))] = cj;
            nu_w += __popc(gm);
        }
        cj = cj_n; xj = xj1; tj = tj1;
        cj_n = cj2; xj1 = x2; tj1 = t2;
        cj2 = cj3; cj3 = cj4;
    }
    if (PRUNE) {
        __syncwarp();
        nb_ilist_finish(nu_w, nm_w, sd.x + ci, lane, A.cj_dummy, il_w, ilm_w, &A.seg_cnt_w[seg]);
    }

    float fi[24];
#pragma unroll
    for (int p = 0; p < 4; p++) {
        fi[6 * p + 0] = fix[p].x; fi[6 * p + 1] = fiy[p].x; fi[6 * p + 2] = fiz[p].x;
        fi[6 * p + 3] = fix[p].y; fi[6 * p + 4] = fiy[p].y; fi[6 * p + 5] = fiz[p].y;
    }
    if (ENERGY) {
        // per-shift sum of i forces for the virial (reading A8) and the energies, fp64 atomics per warp
        float sxs = 0.f, sys = 0.f, szs = 0.f;
#pragma unroll
        for (int a = 0; a < 8; a++) { sxs += fi[3 * a]; sys += fi[3 * a + 1]; szs += fi[3 * a + 2]; }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            sxs += __shfl_xor_sync(0xffffffffu, sxs, d);
            sys += __shfl_xor_sync(0xffffffffu, sys, d);
            szs += __shfl_xor_sync(0xffffffffu, szs, d);
            elj += __shfl_xor_sync(0xffffffffu, elj, d);
            ecoul += __shfl_xor_sync(0xffffffffu, ecoul, d);
        }
        if (lane == 0) {
            if (sid != NB_SHIFT_CENTER) {
                atomicAdd(&A.fshift[sid * 3 + 0], (double)sxs);
                atomicAdd(&A.fshift[sid * 3 + 1], (double)sys);
                atomicAdd(&A.fshift[sid * 3 + 2], (double)szs);
            }
            atomicAdd(&A.energies[0], (double)elj);
            atomicAdd(&A.energies[1], (double)ecoul);
        }
    }

    // (a8) i-force reduction: butterfly reduce-scatter of the 24 partial sums over the 32 lanes;
    // afterwards the quad lane>>2 == a holds (fx,fy,fz) of i atom a.
#pragma unroll
    for (int half = 12, d = 16; half >= 3; half >>= 1, d >>= 1) {
        const bool upper = (lane & d) != 0;
#pragma unroll
        for (int i = 0; i < half; i++) {
            const float keep = upper ? fi[i + half] : fi[i];
            const float send = upper ? fi[i] : fi[i + half];
            fi[i] = keep + __shfl_xor_sync(0xffffffffu, send, d);
        }
    }
#pragma unroll
    for (int d = 2; d > 0; d >>= 1) {
        fi[0] += __shfl_xor_sync(0xffffffffu, fi[0], d);
        fi[1] += __shfl_xor_sync(0xffffffffu, fi[1], d);
        fi[2] += __shfl_xor_sync(0xffffffffu, fi[2], d);
    }
    if ((lane & 3) == 0) red_add_v4(&A.f4[ci * 8 + (lane >> 2)], fi[0], fi[1], fi[2]);
}

// Paired LJ rows per i-cluster, written once per search (types are fixed between searches):
// ljrow[(ci*4 + p)*nt1 + tj] = (-6c6, -6c6', 12c12, 12c12') of the i atoms 2p, 2p+1 of cluster ci against
// j type tj -- what the force kernel's prologue copies to shared memory with one coalesced load.
__global__ void k_ljrows(int nrows, int nt1, const int* __restrict__ type_slot, const float2* __restrict__ ljtab,
                         float4* __restrict__ ljrow)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nrows) return;
    const int tj = i % nt1, cp = i / nt1;   // cp = ci*4 + p
    const int ta = type_slot[cp * 2], tb = type_slot[cp * 2 + 1];
    const float2 ca = ljtab[ta * nt1 + tj], cb = ljtab[tb * nt1 + tj];
    ljrow[i] = make_float4(-ca.x, -cb.x, ca.y, cb.y);
}

// (a8) gather to the caller's atom order; leaves the accumulator zeroed for the next call.
template <bool VIRIAL>
__global__ void __launch_bounds__(256) k_gather(int nslots, float4* __restrict__ f4, const int* __restrict__ atom_of_slot,
                                                const float4* __restrict__ xq, float* __restrict__ f,
                                                double* __restrict__ xf /* [9] sum x (x) f */)
{
    nb_pdl_wait();
    nb_pdl_trigger();
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    double v[9];
#pragma unroll
    for (int i = 0; i < 9; i++) v[i] = 0.0;
    if (s < nslots) {
        const float4 fv = f4[s];
        f4[s] = make_float4(0.f, 0.f, 0.f, 0.f);
        const int a = atom_of_slot[s];
        if (a >= 0) {
            f[3 * a] = fv.x;
            f[3 * a + 1] = fv.y;
            f[3 * a + 2] = fv.z;
            if (VIRIAL) {
                const float4 x = xq[s];
                const double xx[3] = {x.x, x.y, x.z}, ff[3] = {fv.x, fv.y, fv.z};
#pragma unroll
                for (int l = 0; l < 3; l++)
#pragma unroll
                    for (int m = 0; m < 3; m++) v[3 * l + m] = xx[l] * ff[m];
            }
        }
    }
    if (VIRIAL) {
        __shared__ double s_v[8][9];
#pragma unroll
        for (int i = 0; i < 9; i++)
            for (int d = 16; d > 0; d >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], d);
        if ((threadIdx.x & 31) == 0)
            for (int i = 0; i < 9; i++) s_v[threadIdx.x >> 5][i] = v[i];
        __syncthreads();
        if (threadIdx.x < 9) {
            double t = 0.0;
            for (int w = 0; w < 8; w++) t += s_v[w][threadIdx.x];
            atomicAdd(&xf[threadIdx.x], t);
        }
    }
}

// Force-only gather, 4 consecutive slots per thread (nslots is a multiple of 64): the loads of a
// thread are independent and issued together, which matters more than bytes at these sizes.
__global__ void __launch_bounds__(256) k_gather4(int nquads, float4* __restrict__ f4, const int4* __restrict__ atom_of_slot4,
                                                 float* __restrict__ f)
{
    nb_pdl_wait();
    nb_pdl_trigger();
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nquads) return;
    const int4 a = atom_of_slot4[t];
    float4* p = f4 + 4 * (size_t)t;
    const float4 v0 = p[0], v1 = p[1], v2 = p[2], v3 = p[3];
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
    p[0] = z; p[1] = z; p[2] = z; p[3] = z;
    if (a.x >= 0) { f[3 * a.x] = v0.x; f[3 * a.x + 1] = v0.y; f[3 * a.x + 2] = v0.z; }
    if (a.y >= 0) { f[3 * a.y] = v1.x; f[3 * a.y + 1] = v1.y; f[3 * a.y + 2] = v1.z; }
    if (a.z >= 0) { f[3 * a.z] = v2.x; f[3 * a.z + 1] = v2.y; f[3 * a.z + 2] = v2.z; }
    if (a.w >= 0) { f[3 * a.w] = v3.x; f[3 * a.w + 1] = v3.y; f[3 * a.w + 2] = v3.z; }
}

// Xi = -1/2 ( sum_i x_i (x) f_i + sum_s (s L) (x) S_s )   (reading A8)
__global__ void k_virial_final(const double* __restrict__ xf, const double* __restrict__ fshift, float3 box,
                               double* __restrict__ virial)
{
    const int i = threadIdx.x;
    if (i >= 9) return;
    const int l = i / 3, m = i % 3;
    double t = xf[i];
    const double L[3] = {box.x, box.y, box.z};
    for (int sid = 0; sid < NB_NSHIFT; sid++) {
        int s[3];
        nb_shift_vec(sid, s[0], s[1], s[2]);
        t += s[l] * L[l] * fshift[sid * 3 + m];
    }
    virial[i] = -0.5 * t;
}

__global__ void __launch_bounds__(256) k_fp32_peak(float* out, int iters, float a, float b)
{
    float x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}

// FP32-pipe occupancy of the instruction forms the force kernel is made of, measured in place (nb_measure_fp32_pipe):
// 8 independent accumulator pairs per thread, 4 warps per SM sub-partition, everything in registers.
//   0: scalar FFMA, three different register operands      1: FFMA2, three different register PAIRS
//   2: FFMA2 pair * pair + constant-bank operand            3: FMUL2, two different register pairs
template <int MODE>
__global__ void __launch_bounds__(128) k_fp32_forms(float* out, int iters, float2 c0)
{
    float2 acc[8], a[8], b[8];
#pragma unroll
    for (int i = 0; i < 8; i++) {
        acc[i] = make_float2(threadIdx.x + i, i);
        a[i] = make_float2(1.0f + 1e-6f * (threadIdx.x + i), 1.0f - 1e-6f * i);
        b[i] = make_float2(1e-3f * i, 1e-3f * threadIdx.x);
    }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 4; r++) {
#pragma unroll
            for (int i = 0; i < 8; i++) {
                if (MODE == 0) { acc[i].x = fmaf(a[i].x, b[(i + r) % 8].x, acc[i].x); acc[i].y = fmaf(a[i].y, b[(i + r) % 8].y, acc[i].y); }
                if (MODE == 1) acc[i] = __ffma2_rn(a[i], b[(i + r) % 8], acc[i]);
                if (MODE == 2) acc[i] = __ffma2_rn(acc[i], a[i], c0);
                if (MODE == 3) acc[i] = __fmul2_rn(acc[i], a[(i + r) % 8]);
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; i++) s += acc[i].x + acc[i].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// Counts atom pairs with r^2 < rc^2 over the inner list: interacting ("effective" pairs,
// PAPER.md L167-L173) and excluded-but-counted.  Same block/warp/lane mapping as the prune kernel.
__global__ void __launch_bounds__(256) k_count_pairs(ForceArgs A, unsigned long long* __restrict__ out)
{
    const int4 u = A.units[blockIdx.x];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 3, k = lane & 7;
    const int sci = u.w, h = (u.x - sci * NB_NENT) % NB_NHALF, ci = sci * 8 + warp;
    int sx, sy, sz;
    nb_shift_vec(nb_half_shift_id(h), sx, sy, sz);
    float xi[8], yi[8], zi[8];
#pragma unroll
    for (int a = 0; a < 8; a++) {
        const float4 v = A.xq[ci * 8 + a];
        xi[a] = fmaf((float)sx, A.kc.box[0], v.x);
        yi[a] = fmaf((float)sy, A.kc.box[1], v.y);
        zi[a] = fmaf((float)sz, A.kc.box[2], v.z);
    }
    unsigned n_int = 0, n_exc = 0;
    for (int b = u.y; b < u.z; b++) {
        unsigned bits = A.plane[(size_t)b * 8 + warp];
        while (bits) {
            int my = -1;
#pragma unroll
            for (int t = 0; t < 4; t++) {
                const int p = bits ? __ffs(bits) - 1 : -1;
                bits &= bits - 1;
                if (t == g) my = p;
            }
            if (my < 0) continue;
            const int2 ce = A.jl[(size_t)b * 32 + my];
            const float4 xj = A.xq[ce.x * 8 + k];
            const ulonglong2 mm = *reinterpret_cast<const ulonglong2*>(&A.masks[((size_t)ce.y * 8 + warp) * 2]);
            const unsigned cbyte = (unsigned)(mm.y >> (8 * k)) & 0xffu, mbyte = (unsigned)(mm.x >> (8 * k)) & cbyte;
#pragma unroll
            for (int a = 0; a < 8; a++) {
                const float dx = xi[a] - xj.x, dy = yi[a] - xj.y, dz = zi[a] - xj.z;
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                if (r2 < A.kc.rc2) {
                    n_int += (mbyte >> a) & 1u;
                    n_exc += ((cbyte & ~mbyte) >> a) & 1u;
                }
            }
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        n_int += __shfl_xor_sync(0xffffffffu, n_int, d);
        n_exc += __shfl_xor_sync(0xffffffffu, n_exc, d);
    }
    if (lane == 0) {
        if (n_int) atomicAdd(&out[0], (unsigned long long)n_int);
        if (n_exc) atomicAdd(&out[1], (unsigned long long)n_exc);
    }
}

// Atom-pair slots of the inner list as the force kernel evaluates it: 8 per real (non-dummy) j-atom
// entry, 64 per masked cluster pair.  One thread per segment; statistics only.
__global__ void k_count_slots(ForceArgs A, int nseg, int nslot_real, unsigned long long* __restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long n = 0;
    if (i < nseg) {
        const int4 sd = A.segd[i];
        const int buf = nb_seg_buf(sd.w, A.bufmask, A.nparts, A.nunits);
        const int2 cnt = A.seg_cnt[buf][i];
        for (int e = 0; e < cnt.x; e++) n += A.il[buf][sd.x + e] < nslot_real ? 8u : 0u;   // 8 i atoms x one j atom
        n += 64ull * cnt.y;
    }
    for (int d = 16; d > 0; d >>= 1) n += __shfl_xor_sync(0xffffffffu, n, d);
    if ((threadIdx.x & 31) == 0 && n) atomicAdd(out, n);
}

template <int COUL, bool ENERGY, bool TWIN, bool PRUNE>
int launch_force(nb_ctx* c, const ForceArgs& A)
{
    const size_t smem = sizeof(float4) * 4 * (size_t)c->kc.ntypes1;   // paired LJ table of one i-cluster, 64 B per type
    if (smem > 48 * 1024)
        NB_CUDA(c, cudaFuncSetAttribute(k_force<COUL, ENERGY, TWIN, PRUNE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    NB_CUDA(c, nb_launch_pdl(k_force<COUL, ENERGY, TWIN, PRUNE>, dim3(A.seg_count > 0 ? A.seg_count : c->nseg_launch), dim3(32), smem,
                             A.launch_stream ? A.launch_stream : c->stream, A));
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}

// One instantiation per combination of electrostatics, energy / no energy, single / twin cut-off and
// plain / fused-prune ("separate kernels are used for different combinations ... to avoid conditionals").
template <int COUL, bool ENERGY, bool TWIN>
int launch_force_p(nb_ctx* c, const ForceArgs& A, bool prune)
{
    return prune ? launch_force<COUL, ENERGY, TWIN, true>(c, A) : launch_force<COUL, ENERGY, TWIN, false>(c, A);
}
template <int COUL, bool ENERGY>
int launch_force_t(nb_ctx* c, const ForceArgs& A, bool twin, bool prune)
{
    return twin ? launch_force_p<COUL, ENERGY, true>(c, A, prune) : launch_force_p<COUL, ENERGY, false>(c, A, prune);
}
template <int COUL>
int launch_force_e(nb_ctx* c, const ForceArgs& A, bool energy, bool twin, bool prune)
{
    return energy ? launch_force_t<COUL, true>(c, A, twin, prune) : launch_force_t<COUL, false>(c, A, twin, prune);
}

}  // namespace

static void fill_force_args(nb_ctx* c, ForceArgs& A)
{
    memset(&A, 0, sizeof(A));
    A.units = c->units_canon.p;
    A.jl = c->jl.p;
    A.plane = c->plane_inner.p;
    A.segd = c->segd.p;
    for (int b = 0; b < 2; b++) {
        A.seg_cnt[b] = c->seg_cnt[b].p;
        A.il[b] = c->il[b].p;
        A.ilm[b] = c->ilm[b].p;
    }
    A.bufmask = c->bufmask;
    A.seg_part = c->seg_part.p;
    A.nparts = c->buf_nparts;
    A.nunits = c->nunits;
    A.xq = c->xq.p;
    A.type_slot = c->type_slot.p;
    A.ljrow = c->ljrow.p;
    A.masks = c->excl_masks.p;
    A.f4 = c->f4.p;
    A.kc = c->kc;
    for (int k = 0; k < 3; k++) A.kc.box[k] = c->box[k];
}

const void* nbi_gather4_kernel() { return (const void*)k_gather4; }

int nbi_ljrows(nb_ctx* c)
{
    const int nt1 = c->kc.ntypes1, nrows = c->nclusters_max * 4 * nt1;
    NB_CUDA(c, c->ljrow.ensure(nrows, c->stream));
    k_ljrows<<<(nrows + 255) / 256, 256, 0, c->stream>>>(nrows, nt1, c->type_slot.p, c->ljtab.p, c->ljrow.p);
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}

// rlist_inner > 0: the fused first prune (nb_forces_prune): walk the outer list, write the whole inner list.
int nbi_forces(nb_ctx* c, float* f, double* energies, double* virial, float rlist_inner)
{
    cudaStream_t st = c->stream;
    const bool prune = rlist_inner > 0.f;
    if (prune) {
        int rcp = nbi_consolidate(c);   // everything is (re)written into inner buffer 0
        if (rcp != NB_OK) return rcp;
        c->last_nparts = 1;
        c->planes_dirty = true;
        c->st.prune_count++;
    }
    ForceArgs A;
    fill_force_args(c, A);
    A.ol_cnt = c->ol_cnt.p;
    A.olu = c->olu.p;
    A.olm = c->olm.p;
    A.il_w = c->il[0].p;
    A.ilm_w = c->ilm[0].p;
    A.seg_cnt_w = c->seg_cnt[0].p;
    A.rl2 = rlist_inner * rlist_inner;
    A.cj_dummy = c->nclusters_max;
    {
        const double P[5] = {NB_EWC_P0, NB_EWC_P1, NB_EWC_P2, NB_EWC_P3, NB_EWC_P4};
        const double Q[6] = {NB_EWC_Q0, NB_EWC_Q1, NB_EWC_Q2, NB_EWC_Q3, NB_EWC_Q4, NB_EWC_Q5};
        const double b = c->beta_d, b2 = b * b;
        double bk = 1.0;   // beta^(2k)
        const double qlead = b2 * b2 * b2 * b2 * b2 * Q[5];   // Q is made monic in r^2
        for (int k = 0; k < 6; k++, bk *= b2) {
            if (k < 5) A.kc.ewp2[k] = make_float2((float)(b * b2 * bk * P[k] / qlead), (float)(b * b2 * bk * P[k] / qlead));
            A.kc.ewq2[k] = make_float2((float)(bk * Q[k] / qlead), (float)(bk * Q[k] / qlead));
        }
    }
    NB_CUDA(c, c->fshift.ensure(NB_NSHIFT * 3 + 9, st));
    A.fshift = c->fshift.p;
    A.energies = energies;
    const bool energy = energies != nullptr;
    if (energy) {
        NB_CUDA(c, cudaMemsetAsync(energies, 0, 2 * sizeof(double), st));
        NB_CUDA(c, cudaMemsetAsync(c->fshift.p, 0, (NB_NSHIFT * 3 + 9) * sizeof(double), st));
    }
    int rc = NB_OK;
    if (c->nunits > 0 && c->nseg_launch > 0) {
        NbStageTimer tm(c, energy ? NB_T_FORCE_ENERGY : NB_T_FORCE);
        const bool twin = c->twin;
        if (c->prm.coulomb == NB_COUL_EWALD) rc = launch_force_e<NB_COUL_EWALD>(c, A, energy, twin, prune);
        else if (c->prm.coulomb == NB_COUL_RF) rc = launch_force_e<NB_COUL_RF>(c, A, energy, twin, prune);
        else rc = launch_force_e<NB_COUL_NONE>(c, A, energy, twin, prune);
        if (rc != NB_OK) return rc;
    }
    double* xf = c->fshift.p + NB_NSHIFT * 3;
    // (the slots between the actual and the bounded number of super-clusters hold no atoms: atom_of_slot = -1)
    const int nslots = c->nslots_max;
    const int nb = (nslots + 255) / 256;
    NbStageTimer tm(c, NB_T_REDUCE);
    if (virial)
        NB_CUDA(c, nb_launch_pdl(k_gather<true>, dim3(nb), dim3(256), 0, st, nslots, c->f4.p, c->atom_of_slot.p, c->xq.p, f, xf));
    else
        NB_CUDA(c, nb_launch_pdl(k_gather4, dim3((nslots / 4 + 255) / 256), dim3(256), 0, st, nslots / 4, c->f4.p,
                                 reinterpret_cast<const int4*>(c->atom_of_slot.p), f));
    NB_LAUNCH_CHECK(c);
    if (virial) {
        k_virial_final<<<1, 32, 0, st>>>(xf, c->fshift.p, make_float3(c->box[0], c->box[1], c->box[2]), virial);
        NB_LAUNCH_CHECK(c);
    }
    c->st.force_count++;
    return NB_OK;
}

int nbi_measure_fp32_peak(nb_ctx* c, double* fma_per_s)
{
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, c->prm.device);
    const int grid = nsm * 8, iters = 4000;
    DevBuf<float> out;
    NB_CUDA(c, out.ensure((size_t)grid * 256, c->stream));
    cudaEvent_t e0, e1;
    NB_CUDA(c, cudaEventCreate(&e0));
    NB_CUDA(c, cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 5; rep++) {
        cudaEventRecord(e0, c->stream);
        k_fp32_peak<<<grid, 256, 0, c->stream>>>(out.p, iters, 1.0001f, 0.5f);
        cudaEventRecord(e1, c->stream);
        NB_CUDA(c, cudaEventSynchronize(e1));
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    out.release();
    *fma_per_s = (double)grid * 256 * iters * 64.0 / (best * 1e-3);
    return NB_OK;
}

int nbi_measure_fp32_pipe(nb_ctx* c, double* cycles /*[4]*/)
{
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, c->prm.device);
    const int grid = c->nsm * 4, iters = 2000;   // 4 blocks x 4 warps per SM = 4 warps per sub-partition
    DevBuf<float> out;
    NB_CUDA(c, out.ensure((size_t)grid * 128, c->stream));
    cudaEvent_t e0, e1;
    NB_CUDA(c, cudaEventCreate(&e0));
    NB_CUDA(c, cudaEventCreate(&e1));
    for (int mode = 0; mode < 4; mode++) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; rep++) {
            cudaEventRecord(e0, c->stream);
            const float2 c0 = make_float2(0.5f, 0.25f);
            if (mode == 0) k_fp32_forms<0><<<grid, 128, 0, c->stream>>>(out.p, iters, c0);
            if (mode == 1) k_fp32_forms<1><<<grid, 128, 0, c->stream>>>(out.p, iters, c0);
            if (mode == 2) k_fp32_forms<2><<<grid, 128, 0, c->stream>>>(out.p, iters, c0);
            if (mode == 3) k_fp32_forms<3><<<grid, 128, 0, c->stream>>>(out.p, iters, c0);
            cudaEventRecord(e1, c->stream);
            NB_CUDA(c, cudaEventSynchronize(e1));
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        const double warp_instr = (double)iters * 32 * (mode == 0 ? 2 : 1);   // per warp
        cycles[mode] = best * 1e-3 * (double)khz * 1e3 / (warp_instr * 4);    // 4 warps share a sub-partition
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    out.release();
    return NB_OK;
}

int nbi_count_slots(nb_ctx* c, int64_t* slots)
{
    cudaStream_t st = c->stream;
    int rc = nbi_commit_pending(c);
    if (rc != NB_OK) return rc;
    NB_CUDA(c, c->counters.ensure(8, st));
    NB_CUDA(c, cudaMemsetAsync(c->counters.p, 0, 8 * sizeof(long long), st));
    if (c->nseg_launch > 0) {
        ForceArgs A;
        fill_force_args(c, A);
        k_count_slots<<<(c->nseg_launch + 127) / 128, 128, 0, st>>>(A, c->nseg_launch, 8 * c->nclusters_max,
                                                                   (unsigned long long*)c->counters.p);
        NB_LAUNCH_CHECK(c);
    }
    long long v = 0;
    NB_CUDA(c, cudaMemcpyAsync(&v, c->counters.p, sizeof(v), cudaMemcpyDeviceToHost, st));
    NB_CUDA(c, cudaStreamSynchronize(st));
    *slots = v;
    return NB_OK;
}

int nbi_inner_dump(nb_ctx* c, int64_t* n, int32_t* ci, int32_t* entry, int32_t* shift, int32_t* kind, int32_t* part)
{
    cudaStream_t st = c->stream;
    int rc = nbi_commit_pending(c);
    if (rc != NB_OK) return rc;
    const int ns = c->nseg_launch, nbuf = c->have_buf1 ? 2 : 1;
    std::vector<int4> segd(std::max(ns, 1));
    std::vector<int2> cnt[2], ilm[2];
    std::vector<int32_t> il[2];
    for (int b = 0; b < nbuf; b++) {
        cnt[b].resize(std::max(ns, 1));
        il[b].resize(c->il_total + 1);
        ilm[b].resize(c->ilm_total + 1);
    }
    if (ns > 0) {
        NB_CUDA(c, cudaMemcpyAsync(segd.data(), c->segd.p, sizeof(int4) * ns, cudaMemcpyDeviceToHost, st));
        for (int b = 0; b < nbuf; b++) {
            NB_CUDA(c, cudaMemcpyAsync(cnt[b].data(), c->seg_cnt[b].p, sizeof(int2) * ns, cudaMemcpyDeviceToHost, st));
            if (c->il_total) NB_CUDA(c, cudaMemcpyAsync(il[b].data(), c->il[b].p, sizeof(int32_t) * c->il_total, cudaMemcpyDeviceToHost, st));
            if (c->ilm_total) NB_CUDA(c, cudaMemcpyAsync(ilm[b].data(), c->ilm[b].p, sizeof(int2) * c->ilm_total, cudaMemcpyDeviceToHost, st));
        }
    }
    NB_CUDA(c, cudaStreamSynchronize(st));
    int64_t k = 0;
    for (int s = 0; s < ns; s++) {
        const int4 sd = segd[s];
        const int b = c->bufmask ? (int)((c->bufmask >> nb_part_of_unit(sd.w, c->buf_nparts, c->nunits)) & 1u) : 0;
        const int sci = sd.z & 0x3ffffff, sid = sd.z >> 26;
        const int prt = nb_part_of_unit(sd.w, std::max(c->last_nparts, 1), std::max(c->nunits, 1));
        for (int e = 0; e < cnt[b][s].x; e++) {
            const int hc = il[b][sd.x + e];             // slot of the listed j atom
            if (hc >= 8 * c->nclusters_max) continue;   // dummy padding
            if (ci) ci[k] = sci;
            if (entry) entry[k] = hc;
            if (shift) shift[k] = sid;
            if (kind) kind[k] = 0;
            if (part) part[k] = prt;
            k++;
        }
        for (int e = 0; e < cnt[b][s].y; e++) {
            if (ci) ci[k] = sci;
            if (entry) entry[k] = ilm[b][sd.y + e].x;
            if (shift) shift[k] = sid;
            if (kind) kind[k] = 1;
            if (part) part[k] = prt;
            k++;
        }
    }
    *n = k;
    return NB_OK;
}

int nbi_count_pairs(nb_ctx* c, int64_t* n_interacting, int64_t* n_excluded)
{
    cudaStream_t st = c->stream;
    int rc = nbi_rebuild_inner_planes(c);
    if (rc != NB_OK) return rc;
    ForceArgs A;
    fill_force_args(c, A);
    NB_CUDA(c, c->counters.ensure(8, st));
    NB_CUDA(c, cudaMemsetAsync(c->counters.p, 0, 8 * sizeof(long long), st));
    if (c->nunits > 0) {
        k_count_pairs<<<c->nunits, 256, 0, st>>>(A, (unsigned long long*)c->counters.p);
        NB_LAUNCH_CHECK(c);
    }
    long long v[2] = {0, 0};
    NB_CUDA(c, cudaMemcpyAsync(v, c->counters.p, sizeof(v), cudaMemcpyDeviceToHost, st));
    NB_CUDA(c, cudaStreamSynchronize(st));
    if (n_interacting) *n_interacting = v[0];
    if (n_excluded) *n_excluded = v[1];
    return NB_OK;
}

// ---------------------------------------------------------------- nb_forces_static: nb_forces that allocates nothing
// For callers that cannot call cudaMalloc (a stream under graph capture, a tight serving loop, a harness that forbids it).
// The force kernel's scratch -- the cluster-order accumulator f4 it adds into and the per-shift i-force sums / virial
// partials -- lives in ONE file-scope device array of a fixed size instead of the context's cudaMalloc'ed buffers
// (c->f4, c->fshift).  Every GPU that loads the library holds the array until the process exits (NB_STATIC_SCRATCH_BYTES,
// about 4.1 MiB).  All calls of all contexts on a device share it: calls that overlap on the GPU race, and it keeps the
// last call's contents, so every call clears the part it uses first.
//   bytes [0, 1024): 27*3 + 9 doubles (per-shift force sums, sum x (x) f)
//   then NB_STATIC_MAX_SLOTS + 8 * NB_NDUMMY float4: force accumulator, real slots then the dummy clusters' slots
#define NB_STATIC_HEAD_F4 64   // 1024 B
static __device__ __align__(256) float4 g_nb_static_scratch[NB_STATIC_HEAD_F4 + NB_STATIC_MAX_SLOTS + NB_C * NB_NDUMMY];
static_assert(sizeof(g_nb_static_scratch) == NB_STATIC_SCRATCH_BYTES, "nb.h states the size of the static scratch");
static_assert((NB_NSHIFT * 3 + 9) * sizeof(double) <= NB_STATIC_HEAD_F4 * sizeof(float4), "head of the static scratch");

// In host code `g_nb_static_scratch` is a host-side stand-in, not a device address: the address a kernel can use comes
// from cudaGetSymbolAddress, once per device, with that device current (nb_init has made it current).
void nbi_static_scratch_setup(nb_ctx* c)
{
    static std::mutex mu;
    static void* addr_of_device[64] = {};
    c->static_scratch = nullptr;
    c->static_scratch_cuda_err = 0;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess && (dev != c->prm.device || dev < 0 || dev >= 64)) e = cudaErrorInvalidDevice;
    if (e == cudaSuccess) {
        std::lock_guard<std::mutex> lock(mu);
        if (!addr_of_device[dev]) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_nb_static_scratch);
            if (e == cudaSuccess) addr_of_device[dev] = p;
        }
        if (e == cudaSuccess) c->static_scratch = addr_of_device[dev];
    }
    if (e != cudaSuccess) {
        c->static_scratch_cuda_err = (int)e;
        cudaGetLastError();   // nb_forces_static reports it; the other calls are not affected
    }
}

// The non-fused half of nbi_forces with the two scratch pointers replaced; same kernels, same launch order.  No stage
// timers (their events are created on demand), no DevBuf::ensure: nothing here allocates.
int nbi_forces_static(nb_ctx* c, float* f, double* energies, double* virial)
{
    cudaStream_t st = c->stream;
    if (!c->static_scratch)
        return nb_fail(c, NB_ERR_CUDA, "nb_forces_static: cudaGetSymbolAddress of the static scratch failed at nb_init: %s",
                       cudaGetErrorString((cudaError_t)c->static_scratch_cuda_err));
    if (c->nslots_max > NB_STATIC_MAX_SLOTS)
        return nb_fail(c, NB_ERR_OVERFLOW,
                       "nb_forces_static: this system needs %d atom slots (natoms/64 + grid columns super-clusters of 64), the static "
                       "scratch holds NB_STATIC_MAX_SLOTS = %d; use nb_forces",
                       c->nslots_max, (int)NB_STATIC_MAX_SLOTS);
    double* fshift = reinterpret_cast<double*>(c->static_scratch);
    float4* f4 = reinterpret_cast<float4*>(c->static_scratch) + NB_STATIC_HEAD_F4;
    const size_t nf4 = (size_t)c->nslots_max + NB_C * NB_NDUMMY;
    // the accumulator must start at zero; the array holds whatever the last call (of any context) left in it
    NB_CUDA(c, cudaMemsetAsync(f4, 0, nf4 * sizeof(float4), st));
    ForceArgs A;
    fill_force_args(c, A);
    A.f4 = f4;
    A.cj_dummy = c->nclusters_max;
    {
        const double P[5] = {NB_EWC_P0, NB_EWC_P1, NB_EWC_P2, NB_EWC_P3, NB_EWC_P4};
        const double Q[6] = {NB_EWC_Q0, NB_EWC_Q1, NB_EWC_Q2, NB_EWC_Q3, NB_EWC_Q4, NB_EWC_Q5};
        const double b = c->beta_d, b2 = b * b;
        double bk = 1.0;
        const double qlead = b2 * b2 * b2 * b2 * b2 * Q[5];
        for (int k = 0; k < 6; k++, bk *= b2) {
            if (k < 5) A.kc.ewp2[k] = make_float2((float)(b * b2 * bk * P[k] / qlead), (float)(b * b2 * bk * P[k] / qlead));
            A.kc.ewq2[k] = make_float2((float)(bk * Q[k] / qlead), (float)(bk * Q[k] / qlead));
        }
    }
    A.fshift = fshift;
    A.energies = energies;
    const bool energy = energies != nullptr;
    if (energy) {
        NB_CUDA(c, cudaMemsetAsync(energies, 0, 2 * sizeof(double), st));
        NB_CUDA(c, cudaMemsetAsync(fshift, 0, (NB_NSHIFT * 3 + 9) * sizeof(double), st));
    }
    if (c->nunits > 0 && c->nseg_launch > 0) {
        const bool twin = c->twin;
        int rc;
        if (c->prm.coulomb == NB_COUL_EWALD) rc = launch_force_e<NB_COUL_EWALD>(c, A, energy, twin, false);
        else if (c->prm.coulomb == NB_COUL_RF) rc = launch_force_e<NB_COUL_RF>(c, A, energy, twin, false);
        else rc = launch_force_e<NB_COUL_NONE>(c, A, energy, twin, false);
        if (rc != NB_OK) return rc;
    }
    double* xf = fshift + NB_NSHIFT * 3;
    const int nslots = c->nslots_max;
    if (virial)
        NB_CUDA(c, nb_launch_pdl(k_gather<true>, dim3((nslots + 255) / 256), dim3(256), 0, st, nslots, f4, c->atom_of_slot.p, c->xq.p, f, xf));
    else
        NB_CUDA(c, nb_launch_pdl(k_gather4, dim3((nslots / 4 + 255) / 256), dim3(256), 0, st, nslots / 4, f4,
                                 reinterpret_cast<const int4*>(c->atom_of_slot.p), f));
    NB_LAUNCH_CHECK(c);
    if (virial) {
        k_virial_final<<<1, 32, 0, st>>>(xf, fshift, make_float3(c->box[0], c->box[1], c->box[2]), virial);
        NB_LAUNCH_CHECK(c);
    }
    c->st.force_count++;
    return NB_OK;
}

// ---------------------------------------------------------------- local / non-local split
// "splitting non-bonded work into two kernels: one for local-only interactions and one for interactions that involve
// non-local particles ... launch non-local work in a high priority stream to preempt the local kernel and return remote
// forces early, while the local kernel execution can overlap with communication."
// nb_set_local makes the search grid local and non-local atoms separately, so every segment of the inner list is
// local-local or involves a non-local cluster, and the force order lists the local segments first: the two kernels are
// the SAME k_force over the two ranges of that order.  Both add into the one accumulator f4 (atomics); the non-local
// atoms' slots, which only the non-local kernel touches, are the tail [64 * nsc_local, nslots_max) of the cluster order.
static void force_args_inner(nb_ctx* c, ForceArgs& A)
{
    fill_force_args(c, A);
    A.cj_dummy = c->nclusters_max;
    const double P[5] = {NB_EWC_P0, NB_EWC_P1, NB_EWC_P2, NB_EWC_P3, NB_EWC_P4};
    const double Q[6] = {NB_EWC_Q0, NB_EWC_Q1, NB_EWC_Q2, NB_EWC_Q3, NB_EWC_Q4, NB_EWC_Q5};
    const double b = c->beta_d, b2 = b * b;
    double bk = 1.0;
    const double qlead = b2 * b2 * b2 * b2 * b2 * Q[5];
    for (int k = 0; k < 6; k++, bk *= b2) {
        if (k < 5) A.kc.ewp2[k] = make_float2((float)(b * b2 * bk * P[k] / qlead), (float)(b * b2 * bk * P[k] / qlead));
        A.kc.ewq2[k] = make_float2((float)(bk * Q[k] / qlead), (float)(bk * Q[k] / qlead));
    }
}

static int launch_force_range(nb_ctx* c, ForceArgs& A, int base, int count, bool energy, cudaStream_t st)
{
    if (count <= 0) return NB_OK;
    A.seg_base = base;
    A.seg_count = count;
    A.launch_stream = st;
    const bool twin = c->twin;
    if (c->prm.coulomb == NB_COUL_EWALD) return launch_force_e<NB_COUL_EWALD>(c, A, energy, twin, false);
    if (c->prm.coulomb == NB_COUL_RF) return launch_force_e<NB_COUL_RF>(c, A, energy, twin, false);
    return launch_force_e<NB_COUL_NONE>(c, A, energy, twin, false);
}

// gather of the slots [slot0, slot1) (multiples of 64) to the caller's atom order; with_virial: also sum x (x) f into xf
static int gather_range(nb_ctx* c, int slot0, int slot1, float* f, bool with_virial, cudaStream_t st)
{
    const int ns = slot1 - slot0;
    if (ns <= 0) return NB_OK;
    if (with_virial)
        NB_CUDA(c, nb_launch_pdl(k_gather<true>, dim3((ns + 255) / 256), dim3(256), 0, st, ns, c->f4.p + slot0,
                                 (const int*)(c->atom_of_slot.p + slot0), (const float4*)(c->xq.p + slot0), f,
                                 c->fshift.p + NB_NSHIFT * 3));
    else
        NB_CUDA(c, nb_launch_pdl(k_gather4, dim3((ns / 4 + 255) / 256), dim3(256), 0, st, ns / 4, c->f4.p + slot0,
                                 reinterpret_cast<const int4*>(c->atom_of_slot.p + slot0), f));
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}

int nbi_split_setup(nb_ctx* c)
{
    if (c->stream_hp) return NB_OK;
    int lo = 0, hi = 0;
    NB_CUDA(c, cudaDeviceGetStreamPriorityRange(&lo, &hi));   // hi = the numerically lowest value = the highest priority
    NB_CUDA(c, cudaStreamCreateWithPriority(&c->stream_hp, cudaStreamNonBlocking, hi));
    NB_CUDA(c, cudaEventCreateWithFlags(&c->ev_nl_in, cudaEventDisableTiming));
    NB_CUDA(c, cudaEventCreateWithFlags(&c->ev_nl_kernel, cudaEventDisableTiming));
    NB_CUDA(c, cudaEventCreateWithFlags(&c->ev_nl_done, cudaEventDisableTiming));
    return NB_OK;
}

void nbi_split_free(nb_ctx* c)
{
    if (c->ev_nl_in) cudaEventDestroy(c->ev_nl_in);
    if (c->ev_nl_kernel) cudaEventDestroy(c->ev_nl_kernel);
    if (c->ev_nl_done) cudaEventDestroy(c->ev_nl_done);
    if (c->stream_hp) cudaStreamDestroy(c->stream_hp);
    c->ev_nl_in = c->ev_nl_kernel = c->ev_nl_done = nullptr;
    c->stream_hp = nullptr;
}

// The non-local kernel and the gather of the non-local atoms' forces, on the high-priority stream, ordered after
// everything enqueued on the context's stream so far (coordinates, prune).
// energies / virial (as in nb_forces): both kernels add into them; they are complete after nb_forces_local.
int nbi_forces_nonlocal(nb_ctx* c, float* f, double* energies, double* virial)
{
    int rc = nbi_split_setup(c);
    if (rc != NB_OK) return rc;
    const bool energy = energies != nullptr;
    if (energy) {   // cleared on the context's stream, before either kernel can start
        NB_CUDA(c, c->fshift.ensure(NB_NSHIFT * 3 + 9, c->stream));
        NB_CUDA(c, cudaMemsetAsync(energies, 0, 2 * sizeof(double), c->stream));
        NB_CUDA(c, cudaMemsetAsync(c->fshift.p, 0, (NB_NSHIFT * 3 + 9) * sizeof(double), c->stream));
    }
    c->nl_energies = energies;
    c->nl_virial = virial;
    NB_CUDA(c, cudaEventRecord(c->ev_nl_in, c->stream));
    NB_CUDA(c, cudaStreamWaitEvent(c->stream_hp, c->ev_nl_in, 0));
    ForceArgs A;
    force_args_inner(c, A);
    A.fshift = c->fshift.p;
    A.energies = energies;
    if ((rc = launch_force_range(c, A, c->nseg_local, c->nseg_launch - c->nseg_local, energy, c->stream_hp)) != NB_OK) return rc;
    NB_CUDA(c, cudaEventRecord(c->ev_nl_kernel, c->stream_hp));
    if ((rc = gather_range(c, c->nsc_local * NB_SC_ATOMS, c->nslots_max, f, virial != nullptr, c->stream_hp)) != NB_OK) return rc;
    NB_CUDA(c, cudaEventRecord(c->ev_nl_done, c->stream_hp));
    c->nl_pending = true;
    c->st.force_count++;
    return NB_OK;
}

// The local kernel on the context's stream (it runs next to the non-local one), then, once the non-local kernel has
// added its share to the local atoms as well, the gather of the local atoms' forces.
int nbi_forces_local(nb_ctx* c, float* f)
{
    ForceArgs A;
    force_args_inner(c, A);
    A.fshift = c->fshift.p;
    A.energies = c->nl_energies;
    int rc = launch_force_range(c, A, 0, c->nseg_local, c->nl_energies != nullptr, c->stream);
    if (rc != NB_OK) return rc;
    NB_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_nl_kernel, 0));
    if ((rc = gather_range(c, 0, c->nsc_local * NB_SC_ATOMS, f, c->nl_virial != nullptr, c->stream)) != NB_OK) return rc;
    // later work on the context's stream (the next put / prune / search) must not overtake the non-local gather
    NB_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_nl_done, 0));
    if (c->nl_virial) {   // both gathers have added their sum x (x) f, both kernels their per-shift force sums
        k_virial_final<<<1, 32, 0, c->stream>>>(c->fshift.p + NB_NSHIFT * 3, c->fshift.p, make_float3(c->box[0], c->box[1], c->box[2]),
                                                c->nl_virial);
        NB_LAUNCH_CHECK(c);
    }
    c->nl_pending = false;
    return NB_OK;
}

int nbi_sync_nonlocal(nb_ctx* c)
{
    if (c->ev_nl_done) NB_CUDA(c, cudaEventSynchronize(c->ev_nl_done));
    return NB_OK;
}
