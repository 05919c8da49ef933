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
// j atoms: 4 j-clusters x 8 atoms per step, the 8 i-atoms live in registers.
#include "nb_internal.h"

namespace {

struct PruneArgs {
    const int4* units;
    const int2* jl;
    const uint32_t* plane_outer;
    uint32_t* plane_inner;
    const float4* xq;
    float box[3];
    float rl2;   // fl32(rlist_inner^2), reading A12
};

__global__ void __launch_bounds__(256) k_prune(PruneArgs A)
{
    const int4 u = A.units[blockIdx.x];
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
    for (int b = u.y; b < u.z; b++) {
        unsigned bits = A.plane_outer[(size_t)b * 8 + warp];
        unsigned result = 0;
        while (bits) {
            int p[4];
#pragma unroll
            for (int t = 0; t < 4; t++) {
                p[t] = bits ? __ffs(bits) - 1 : -1;
                bits &= bits - 1;
            }
            const int my = g == 0 ? p[0] : (g == 1 ? p[1] : (g == 2 ? p[2] : p[3]));
            const bool valid = my >= 0;
            const int cj = valid ? A.jl[(size_t)b * 32 + my].x : ci;
            const float4 xj = A.xq[cj * 8 + k];
            const bool diag = cj == ci && h == 0;
            bool found = false;
#pragma unroll
            for (int a = 0; a < 8; a++) {
                const float dx = __fsub_rn(xi[a], xj.x), dy = __fsub_rn(yi[a], xj.y), dz = __fsub_rn(zi[a], xj.z);
                const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                bool ok = d2 < A.rl2;
                if (diag) ok = ok && (k > a);   // zero-shift diagonal: only b > a are pairs
                found = found || ok;
            }
            const unsigned gm = __ballot_sync(0xffffffffu, found && valid);
#pragma unroll
            for (int t = 0; t < 4; t++)
                if (p[t] >= 0 && ((gm >> (8 * t)) & 0xffu)) result |= 1u << p[t];
        }
        if (lane == 0) A.plane_inner[(size_t)b * 8 + warp] = result;
    }
}

}  // namespace

int nbi_prune(nb_ctx* c, float rlist_inner, int part, int nparts)
{
    const long long nu = c->nunits;
    const int u0 = (int)((long long)part * nu / nparts), u1 = (int)((long long)(part + 1) * nu / nparts);
    c->last_nparts = nparts;
    c->st.prune_count++;
    if (u1 <= u0) return NB_OK;
    PruneArgs A;
    A.units = c->units_canon.p + u0;
    A.jl = c->jl.p;
    A.plane_outer = c->plane_outer.p;
    A.plane_inner = c->plane_inner.p;
    A.xq = c->xq.p;
    for (int k = 0; k < 3; k++) A.box[k] = c->box[k];
    A.rl2 = rlist_inner * rlist_inner;
    NbStageTimer tm(c, NB_T_PRUNE);
    k_prune<<<u1 - u0, 256, 0, c->stream>>>(A);
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}
