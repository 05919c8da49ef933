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

// 8 exact (A12) distance checks of this lane's j atom; DIAG keeps only pairs b > a.
template <bool DIAG>
__device__ __forceinline__ bool prune_checks(const float (&xi)[8], const float (&yi)[8], const float (&zi)[8],
                                             const float4 xj, float rl2, bool diag, int k)
{
    bool found = false;
#pragma unroll
    for (int a = 0; a < 8; a++) {
        const float dx = __fsub_rn(xi[a], xj.x), dy = __fsub_rn(yi[a], xj.y), dz = __fsub_rn(zi[a], xj.z);
        const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
        bool ok = d2 < rl2;
        if (DIAG) ok = ok && (!diag || k > a);   // zero-shift diagonal: only b > a are pairs
        found = found || ok;
    }
    return found;
}

__global__ void __launch_bounds__(256) k_prune(PruneArgs A)
{
    __shared__ int2 s_q[8][40];                          // {cj, unit-local joint slot}
    __shared__ unsigned s_res[8][NB_MAX_UNIT_BATCHES];   // inner mask words of this warp's plane
    const int ucan = A.order[blockIdx.x];
    const int4 u = A.units[ucan];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 3, k = lane & 7;
    const int sci = u.w, h = u.x - sci * NB_NHALF, ci = sci * 8 + warp;
    int sx, sy, sz;
    nb_shift_vec(nb_half_shift_id(h), sx, sy, sz);
    float xi[8], yi[8], zi[8];
#pragma unroll
    for (int a = 0; a < 8; a++) {
        const float4 v = A.xq[ci * 8 + a];
        xi[a] = __fmaf_rn((float)sx, A.box[0], v.x);   // A12: t = fmaf(s, L, x_a), one rounding
        yi[a] = __fmaf_rn((float)sy, A.box[1], v.y);
        zi[a] = __fmaf_rn((float)sz, A.box[2], v.z);
    }
    int2* q = s_q[warp];
    unsigned* res = s_res[warp];
    if (lane < NB_MAX_UNIT_BATCHES) res[lane] = 0u;
    const unsigned lt = (1u << lane) - 1u;
    int nq = 0;
    unsigned bits = A.plane_outer[(size_t)u.y * 8 + warp];
    int cje = ((bits >> lane) & 1u) ? A.jl[(size_t)u.y * 32 + lane].x : 0;
    __syncwarp();
    for (int b = u.y; b < u.z; b++) {
        const bool last = b + 1 == u.z;
        unsigned bits_n = 0;
        int cje_n = 0;
        if (!last) {
            bits_n = A.plane_outer[(size_t)(b + 1) * 8 + warp];
            if ((bits_n >> lane) & 1u) cje_n = A.jl[(size_t)(b + 1) * 32 + lane].x;
        }
        if ((bits >> lane) & 1u) q[nq + __popc(bits & lt)] = make_int2(cje, (b - u.y) * 32 + lane);
        nq += __popc(bits);
        __syncwarp();
        int done = 0;
        const int need = last ? 1 : 4;   // the unit's last batch also runs the partly filled step
        if (nq >= need) {
            bool valid = g < nq;
            int2 ce = valid ? q[g] : make_int2(ci, 0);
            float4 xj = A.xq[ce.x * 8 + k];
            while (true) {
                done += 4;
                const bool more = nq - done >= need;
                bool valid_n = false;
                int2 ce_n = ce;
                float4 xj_n = xj;
                if (more) {
                    valid_n = done + g < nq;
                    ce_n = valid_n ? q[done + g] : make_int2(ci, 0);
                    xj_n = A.xq[ce_n.x * 8 + k];
                }
                const bool diag = ce.x == ci && h == 0;
                bool found;
                if (__any_sync(0xffffffffu, diag)) found = prune_checks<true>(xi, yi, zi, xj, A.rl2, diag, k);
                else found = prune_checks<false>(xi, yi, zi, xj, A.rl2, false, k);
                const unsigned gm = __ballot_sync(0xffffffffu, found && valid);
                if (k == 0 && ((gm >> (8 * g)) & 0xffu)) atomicOr(&res[ce.y >> 5], 1u << (ce.y & 31));
                if (!more) break;
                valid = valid_n;
                ce = ce_n;
                xj = xj_n;
            }
            done = min(done, nq);
        }
        const int rem = nq - done;
        int2 t = make_int2(0, 0);
        if (lane < rem) t = q[done + lane];
        __syncwarp();
        if (lane < rem) q[lane] = t;
        __syncwarp();
        nq = rem;
        bits = bits_n;
        cje = cje_n;
    }
    __syncwarp();
    if (lane < u.z - u.y) A.plane_inner[(size_t)(u.y + lane) * 8 + warp] = res[lane];
    int4* sg = &A.seg[A.seg_pos[A.unit_pos[ucan] * 8 + warp]];
    const int2 off = *reinterpret_cast<const int2*>(sg);
    nb_ilist_write([&](int b) { return res[b]; }, u.y, u.z, warp, lane, A.cj_dummy, A.plane_excl, A.jl, A.il + off.x, A.ilm + off.y,
                   reinterpret_cast<int2*>(sg) + 1);
}

}  // namespace

int nbi_prune(nb_ctx* c, float rlist_inner, int part, int nparts)
{
    const long long nu = c->nunits;
    const int u0 = (int)((long long)part * nu / nparts), u1 = (int)((long long)(part + 1) * nu / nparts);
    c->last_nparts = nparts;
    c->st.prune_count++;
    if (u1 <= u0) return NB_OK;
    if (c->prune_order_nparts != nparts || c->prune_order_search != c->st.search_count) {
        // launch order inside each rolling part: longest work unit first, so that the last
        // wave of blocks is made of short units; rebuilt once per search / change of nparts
        c->h_prune_order.resize(nu);
        for (int i = 0; i < nu; i++) c->h_prune_order[i] = i;
        for (int p = 0; p < nparts; p++) {
            const long long a = (long long)p * nu / nparts, b = (long long)(p + 1) * nu / nparts;
            std::stable_sort(c->h_prune_order.begin() + a, c->h_prune_order.begin() + b, [&](int x, int y) {
                return (c->h_units[x].z - c->h_units[x].y) > (c->h_units[y].z - c->h_units[y].y);
            });
        }
        NB_CUDA(c, c->prune_order.ensure(nu, c->stream));
        NB_CUDA(c, cudaMemcpyAsync(c->prune_order.p, c->h_prune_order.data(), sizeof(int) * nu, cudaMemcpyHostToDevice, c->stream));
        c->prune_order_nparts = nparts;
        c->prune_order_search = c->st.search_count;
    }
    PruneArgs A;
    A.units = c->units_canon.p;
    A.order = c->prune_order.p + u0;
    A.jl = c->jl.p;
    A.plane_outer = c->plane_outer.p;
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
    k_prune<<<u1 - u0, 256, 0, c->stream>>>(A);
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}
