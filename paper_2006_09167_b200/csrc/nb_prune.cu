// nb_prune.cu -- (a6) dynamic pruning of the outer list to the inner list, full or rolling.
//
// "A particle-pair distance based list pruning is carried out on the GPU which
// eliminates non-interacting cluster pairs"; L193: dual pair list, "frequent pruning steps
// produce a pair list based on the inner cut-off ... pruning is done in a rolling fashion
// scheduled in chunks between force computations".
//
// The outer masks are never modified; every prune of a part restarts from them (atoms move
// both ways) and rewrites the inner mask words of that part only (reading A15).  Part p of k
// is the contiguous range [p*nu/k, (p+1)*nu/k) of the canonically ordered work units.
// Block = 8 warps = the 8 i-clusters of one super-cluster (one work unit); warp w owns the
// bit-plane w of the unit's mask words, so no cross-warp combination is needed.  Lanes own
// j atoms: 4 j-clusters x 8 atoms per step, the 8 i-atoms live in registers.  The set bits of
// the outer plane words are compacted into a per-warp queue (as in the force kernel), so every
// step but the unit's last is full, and the j coordinates of the next step are loaded before
// the current step's arithmetic.
#include "nb_internal.h"

#include <algorithm>

namespace {

struct PruneArgs {
    const int4* units;        // canonical order
    const int* order;         // launch order of this part: canonical unit indices, longest first
    const int2* jl;
    const uint32_t* plane_outer;
    const int2* ol;           // compact outer list (nb_list.cu k_ilist_build)
    const int2* ol_cnt;
    uint32_t* plane_inner;
    const float4* xq;
    float box[3];
    float rl2;   // fl32(rlist_inner^2), reading A12
    // compact inner list written for the force kernel (nb_internal.h)
    int u0;      // canonical index of units[0]
    int cj_dummy;
    const uint32_t* plane_excl;
    const int* unit_pos;
    const int* seg_pos;
    int4* seg;
    int32_t* il;
    int2* ilm;
};

// 8 exact (A12) distance checks of this lane's j atom against the i atoms (packed pairs 2p, 2p+1:
// the FP32x2 instructions round each half like their scalar forms, and x_a + (-x_b) is x_a - x_b
// exactly, so list parity with the oracle is unchanged); DIAG keeps only pairs b > a.
template <bool DIAG>
__device__ __forceinline__ bool prune_checks(const float2 (&xi)[4], const float2 (&yi)[4], const float2 (&zi)[4],
                                             const float4 xj, float rl2, bool diag, int k)
{
    const float2 nx = make_float2(-xj.x, -xj.x), ny = make_float2(-xj.y, -xj.y), nz = make_float2(-xj.z, -xj.z);
    bool found = false;
#pragma unroll
    for (int p = 0; p < 4; p++) {
        const float2 dx = __fadd2_rn(xi[p], nx), dy = __fadd2_rn(yi[p], ny), dz = __fadd2_rn(zi[p], nz);
        const float2 d2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
        bool ok0 = d2.x < rl2, ok1 = d2.y < rl2;
        if (DIAG) {   // zero-shift diagonal: only b > a are pairs
            ok0 = ok0 && (!diag || k > 2 * p);
            ok1 = ok1 && (!diag || k > 2 * p + 1);
        }
        found = found || ok0 || ok1;
    }
    return found;
}

// One survivor-append step: 4 j-clusters (lane groups), entry e = {cj, unit-local joint slot | masked << 30}.
struct PruneState {
    int nu, nm;
};

// One step over 4 cluster pairs WITHOUT a mask: a half j-cluster (4 atoms) survives iff one of its
// atoms is within rlist_inner of an i atom; the survivors' half-cluster indices are appended to il.
__device__ __forceinline__ void prune_step_unmasked(const PruneArgs& A, const float2 (&xi)[4], const float2 (&yi)[4],
                                                    const float2 (&zi)[4], const int2 e, const float4 x, const bool valid,
                                                    const int lane, unsigned* res, int32_t* il, PruneState& st)
{
    const bool found = prune_checks<false>(xi, yi, zi, x, A.rl2, false, 0);
    const unsigned gm = __ballot_sync(0xffffffffu, found && valid);
    unsigned hm = gm | (gm >> 1);
    hm = (hm | (hm >> 2)) & 0x11111111u;          // bit 4h: half h of the step (lanes 4h..4h+3) has a survivor
    if ((hm >> lane) & 1u) {                      // its leader lane (lane % 4 == 0)
        il[st.nu + __popc(hm & ((1u << lane) - 1u))] = 2 * e.x + ((lane >> 2) & 1);
        if ((lane & 4) == 0 || !((hm >> (lane - 4)) & 1u)) atomicOr(&res[e.y >> 5], 1u << (e.y & 31));   // once per cluster
    }
    st.nu += __popc(hm);
}

// One step over 4 cluster pairs WITH a mask (exclusions, or the zero-shift diagonal pair, which keeps
// only atom pairs b > a): whole clusters, appended to ilm with their mask reference.
__device__ __forceinline__ void prune_step_masked(const PruneArgs& A, const float2 (&xi)[4], const float2 (&yi)[4],
                                                  const float2 (&zi)[4], const int2 e, const float4 x, const bool valid,
                                                  const bool diag, const int b0, const int lane, unsigned* res, int2* ilm,
                                                  PruneState& st)
{
    const int g = lane >> 3, k = lane & 7;
    const bool found = prune_checks<true>(xi, yi, zi, x, A.rl2, diag, k);
    const unsigned gm = __ballot_sync(0xffffffffu, found && valid);
    unsigned cm = gm | (gm >> 1);
    cm |= cm >> 2;
    cm = (cm | (cm >> 4)) & 0x01010101u;          // bit 8g: cluster pair g of the step survives
    if ((cm >> lane) & 1u) {
        atomicOr(&res[e.y >> 5], 1u << (e.y & 31));
        ilm[st.nm + __popc(cm & ((1u << lane) - 1u))] = make_int2(e.x, A.jl[(size_t)b0 * 32 + e.y].y);
    }
    st.nm += __popc(cm);
}

// One warp per block = one i-cluster of one work unit: streams its compact outer list segment.
__global__ void __launch_bounds__(32) k_prune(PruneArgs A)
{
    __shared__ unsigned s_res[NB_MAX_UNIT_BATCHES];   // inner mask words of this i-cluster's plane
    const int sidx = A.order[blockIdx.x];   // canonical unit * 8 + i-cluster, longest list first within the part
    const int ucan = sidx >> 3, warp = sidx & 7;
    const int4 u = A.units[ucan];
    const int lane = threadIdx.x & 31, g = lane >> 3, k = lane & 7;
    const int sci = u.w, h = u.x - sci * NB_NHALF, ci = sci * 8 + warp;
    const int s0 = A.unit_pos[ucan] * 8 + warp;
    int4* sg = &A.seg[A.seg_pos[s0]];
    const int2 off = *reinterpret_cast<const int2*>(sg);
    const int2 n = A.ol_cnt[s0];            // {cluster pairs without a mask, with a mask}
    const int2* __restrict__ ol = A.ol + off.x + off.y;
    int32_t* il = A.il + off.x;
    int2* ilm = A.ilm + off.y;
    const int ns = (n.x + 3) >> 2;
    int2 ea = make_int2(ci, 0), eb = ea, ea2 = ea, eb2 = ea;
    if (ns > 0) {
        ea = ol[min(g, n.x - 1)];
        eb = ol[min(4 + g, n.x - 1)];
        ea2 = ol[min(8 + g, n.x - 1)];
        eb2 = ol[min(12 + g, n.x - 1)];
    }
    int sx, sy, sz;
    nb_shift_vec(nb_half_shift_id(h), sx, sy, sz);
    float2 xi[4], yi[4], zi[4];
#pragma unroll
    for (int p = 0; p < 4; p++) {
        const float4 v0 = A.xq[ci * 8 + 2 * p], v1 = A.xq[ci * 8 + 2 * p + 1];
        // A12: t = fmaf(s, L, x_a), one rounding
        xi[p] = make_float2(__fmaf_rn((float)sx, A.box[0], v0.x), __fmaf_rn((float)sx, A.box[0], v1.x));
        yi[p] = make_float2(__fmaf_rn((float)sy, A.box[1], v0.y), __fmaf_rn((float)sy, A.box[1], v1.y));
        zi[p] = make_float2(__fmaf_rn((float)sz, A.box[2], v0.z), __fmaf_rn((float)sz, A.box[2], v1.z));
    }
    unsigned* res = s_res;
    if (lane < NB_MAX_UNIT_BATCHES) res[lane] = 0u;
    __syncwarp();
    PruneState st = {0, 0};
    // cluster pairs with a mask: few (about one step per zero-shift segment), no pipeline
    const int mbase = (n.x + 3) & ~3;
    for (int s = 0; s < n.y; s += 4) {
        const bool valid = s + g < n.y;
        const int2 e = ol[mbase + min(s + g, n.y - 1)];
        const float4 x = A.xq[e.x * 8 + k];
        prune_step_masked(A, xi, yi, zi, e, x, valid, e.x == ci && h == 0, u.y, lane, res, ilm, st);
    }
    if (ns > 0) {
        // two alternating register sets (a: even steps, b: odd steps); j coordinates two steps ahead,
        // list entries four steps ahead, indices clamped to the segment (as in the force kernel)
        float4 xa = A.xq[ea.x * 8 + k], xb = A.xq[eb.x * 8 + k];
        int s = 0;
        for (; s + 1 < ns; s += 2) {
            prune_step_unmasked(A, xi, yi, zi, ea, xa, 4 * s + g < n.x, lane, res, il, st);
            ea = ea2;
            xa = A.xq[ea.x * 8 + k];
            ea2 = ol[min(4 * (s + 4) + g, n.x - 1)];
            prune_step_unmasked(A, xi, yi, zi, eb, xb, 4 * (s + 1) + g < n.x, lane, res, il, st);
            eb = eb2;
            xb = A.xq[eb.x * 8 + k];
            eb2 = ol[min(4 * (s + 5) + g, n.x - 1)];
        }
        if (s < ns) prune_step_unmasked(A, xi, yi, zi, ea, xa, 4 * s + g < n.x, lane, res, il, st);
    }
    __syncwarp();
    nb_ilist_finish(st.nu, st.nm, u.y * 8 + warp, lane, A.cj_dummy, il, ilm, reinterpret_cast<int2*>(sg) + 1);
    if (lane < u.z - u.y) A.plane_inner[(size_t)(u.y + lane) * 8 + warp] = res[lane];
}

}  // namespace

int nbi_prune(nb_ctx* c, float rlist_inner, int part, int nparts)
{
    const long long nu = c->nunits;
    const int u0 = (int)((long long)part * nu / nparts), u1 = (int)((long long)(part + 1) * nu / nparts);
    c->last_nparts = nparts;
    c->st.prune_count++;
    if (u1 <= u0) return NB_OK;
    // Launch order inside each rolling part: longest i-cluster list first, so that the last
    // wave of blocks is made of short lists.  Derived in one pass from the force kernel's global
    // longest-first order (made at search time); cached per nparts until the next search.
    nb_ctx::PruneOrder* po = nullptr;
    for (auto& e : c->prune_orders)
        if (e.nparts == nparts && e.search == c->st.search_count) po = &e;
    if (!po) {
        po = &c->prune_orders[c->prune_order_next];
        c->prune_order_next = (c->prune_order_next + 1) % 4;
        std::vector<int32_t> fill(nparts), part_of(nu);
        for (int p = 0; p < nparts; p++) {
            const long long a = (long long)p * nu / nparts, b = (long long)(p + 1) * nu / nparts;
            fill[p] = (int)(a * 8);
            for (long long i = a; i < b; i++) part_of[i] = p;
        }
        po->h.resize(nu * 8);
        for (long long t = 0; t < nu * 8; t++) {
            const int s0 = c->h_seg_sorted[t], ucan = c->h_unit_order[s0 >> 3];
            po->h[fill[part_of[ucan]]++] = ucan * 8 + (s0 & 7);
        }
        NB_CUDA(c, po->d.ensure(nu * 8, c->stream));
        NB_CUDA(c, cudaMemcpyAsync(po->d.p, po->h.data(), sizeof(int) * nu * 8, cudaMemcpyHostToDevice, c->stream));
        po->nparts = nparts;
        po->search = c->st.search_count;
    }
    PruneArgs A;
    A.units = c->units_canon.p;
    A.order = po->d.p + (size_t)u0 * 8;
    A.jl = c->jl.p;
    A.plane_outer = c->plane_outer.p;
    A.ol = c->ol.p;
    A.ol_cnt = c->ol_cnt.p;
    A.plane_inner = c->plane_inner.p;
    A.xq = c->xq.p;
    for (int k = 0; k < 3; k++) A.box[k] = c->box[k];
    A.rl2 = rlist_inner * rlist_inner;
    A.u0 = u0;
    A.cj_dummy = c->nclusters;
    A.plane_excl = c->plane_excl.p;
    A.unit_pos = c->unit_pos.p; A.seg_pos = c->seg_pos.p; A.seg = c->seg.p;
    A.il = c->il.p; A.ilm = c->ilm.p;
    NbStageTimer tm(c, NB_T_PRUNE);
    k_prune<<<(u1 - u0) * 8, 32, 0, c->stream>>>(A);
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}
