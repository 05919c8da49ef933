// nb_prune.cu -- (a6) dynamic pruning of the outer list to the inner list, full or rolling.
//
// "A particle-pair distance based list pruning is carried out on the GPU which
// eliminates non-interacting cluster pairs"; L193: dual pair list, "frequent pruning steps
// produce a pair list based on the inner cut-off ... pruning is done in a rolling fashion
// scheduled in chunks between force computations ... which allows it to overlap other work".
//
// The outer list is never modified; every prune of a part restarts from it (atoms move both ways)
// and rewrites the inner list segments of that part only (reading A15).  Part p of k is the
// contiguous range [p*nu/k, (p+1)*nu/k) of the canonically ordered work units.
// One thread block = one warp = one SEGMENT (one i-cluster of one work unit): it streams the
// segment's compact outer list (nb_list.cu k_ilist_build: plain cj for the cluster pairs without a
// mask, {cj, mask ref} for those with one), 4 j-clusters per step, lanes own j atoms, the 8 i atoms
// live in registers as packed pairs; ONE ballot per step gives the surviving halves (or clusters),
// which the leader lanes append to the inner list segment the force kernel streams.
//
// Two ways to schedule it: nb_prune enqueues the kernel on the context's stream (the next nb_forces
// sees its result); nb_prune_overlapped runs it on a second stream next to the force kernel of the
// same step, writing into the inner-list buffer the force kernel is not reading; the part flips to the
// new buffer at the next nb_put_atoms.
#include "nb_internal.h"

#include <algorithm>

namespace {

struct PruneArgs {
    const int* order;         // launch order of this part: segment ids, longest outer list first
    const int4* segd;
    const int2* ol_cnt;
    const int32_t* olu;       // compact outer list (nb_list.cu k_ilist_build)
    const int2* olm;
    const float4* xq;
    float box[3];
    float rl2;                // fl32(rlist_inner^2), reading A12
    int cj_dummy;
    // inner list written for the force kernel (nb_internal.h): buffer `wbuf` when the segment's part bit says so
    int32_t* il[2];
    int2* ilm[2];
    int2* seg_cnt[2];
    int wb;                   // inner buffer this part is written into (all segments of a launch belong to one part)
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

// One step over 4 cluster pairs WITHOUT a mask: a j atom survives iff it is within rlist_inner of an i atom; the
// survivors' slot indices are appended to il in lane order (one ballot, one popc per lane).
__device__ __forceinline__ void prune_step_unmasked(const float2 (&xi)[4], const float2 (&yi)[4], const float2 (&zi)[4],
                                                    const float rl2, const int cj, const float4 x, const bool valid,
                                                    const int lane, int32_t* __restrict__ il, int& nu)
{
    const bool found = prune_checks<false>(xi, yi, zi, x, rl2, false, 0) && valid;
    const unsigned gm = __ballot_sync(0xffffffffu, found);
    if (found) il[nu + __popc(gm & ((1u << lane) - 1u))] = cj * 8 + (lane & 7);
    nu += __popc(gm);
}

// One step over 4 cluster pairs WITH a mask (exclusions, or the zero-shift diagonal pair, which keeps
// only atom pairs b > a): whole clusters, appended to ilm with their mask reference.
__device__ __forceinline__ void prune_step_masked(const float2 (&xi)[4], const float2 (&yi)[4], const float2 (&zi)[4],
                                                  const float rl2, const int2 e, const float4 x, const bool valid,
                                                  const bool diag, const int lane, int2* __restrict__ ilm, int& nm)
{
    const int k = lane & 7;
    const bool found = prune_checks<true>(xi, yi, zi, x, rl2, diag, k);
    const unsigned gm = __ballot_sync(0xffffffffu, found && valid);
    unsigned cm = gm | (gm >> 1);
    cm |= cm >> 2;
    cm = (cm | (cm >> 4)) & 0x01010101u;          // bit 8g: cluster pair g of the step survives
    if ((cm >> lane) & 1u) ilm[nm + __popc(cm & ((1u << lane) - 1u))] = e;
    nm += __popc(cm);
}

// One warp per block = one segment: streams its compact outer list.
__global__ void __launch_bounds__(32) k_prune(PruneArgs A)
{
    nb_pdl_wait();
    nb_pdl_trigger();
    const int t = A.order[blockIdx.x];
    const int2 n = A.ol_cnt[t];             // {cluster pairs without a mask, with a mask}
    if (n.x + n.y == 0) return;             // (an empty outer segment has an empty inner one, set at search time)
    const int4 sd = A.segd[t];
    const int lane = threadIdx.x & 31, g = lane >> 3, k = lane & 7;
    const int ci = sd.z & 0x3ffffff, sid = sd.z >> 26;
    const int wb = A.wb;
    const int32_t* __restrict__ olu = A.olu + sd.x;
    const int2* __restrict__ olm = A.olm + sd.y;
    // (selected, not indexed: a run-time index into the kernel parameters makes ptxas copy them to local memory)
    int32_t* il = (wb ? A.il[1] : A.il[0]) + sd.x;
    int2* ilm = (wb ? A.ilm[1] : A.ilm[0]) + sd.y;
    const int ns = (n.x + 3) >> 2;
    int ea = ci, eb = ci, ea2 = ci, eb2 = ci;
    if (ns > 0) {
        ea = olu[min(g, n.x - 1)];
        eb = olu[min(4 + g, n.x - 1)];
        ea2 = olu[min(8 + g, n.x - 1)];
        eb2 = olu[min(12 + g, n.x - 1)];
    }
    int sx, sy, sz;
    nb_shift_vec(sid, sx, sy, sz);
    float2 xi[4], yi[4], zi[4];
#pragma unroll
    for (int p = 0; p < 4; p++) {
        const float4 v0 = A.xq[ci * 8 + 2 * p], v1 = A.xq[ci * 8 + 2 * p + 1];
        // A12: t = fmaf(s, L, x_a), one rounding
        xi[p] = make_float2(__fmaf_rn((float)sx, A.box[0], v0.x), __fmaf_rn((float)sx, A.box[0], v1.x));
        yi[p] = make_float2(__fmaf_rn((float)sy, A.box[1], v0.y), __fmaf_rn((float)sy, A.box[1], v1.y));
        zi[p] = make_float2(__fmaf_rn((float)sz, A.box[2], v0.z), __fmaf_rn((float)sz, A.box[2], v1.z));
    }
    int nu = 0, nm = 0;
    // two alternating register sets (a: even steps, b: odd steps); j coordinates two steps ahead,
    // list entries four steps ahead, indices clamped to the segment (as in the force kernel); the first two
    // coordinate loads are in flight during the masked steps
    float4 xa = make_float4(0.f, 0.f, 0.f, 0.f), xb = xa;
    if (ns > 0) {
        xa = A.xq[ea * 8 + k];
        xb = A.xq[eb * 8 + k];
    }
    // cluster pairs with a mask: few (about one step per zero-shift segment), no pipeline
    for (int s = 0; s < n.y; s += 4) {
        const bool valid = s + g < n.y;
        const int2 e = olm[min(s + g, n.y - 1)];
        const float4 x = A.xq[e.x * 8 + k];
        prune_step_masked(xi, yi, zi, A.rl2, e, x, valid, e.x == ci && sid == NB_SHIFT_CENTER, lane, ilm, nm);
    }
    if (ns > 0) {
        int s = 0;
        for (; s + 1 < ns; s += 2) {
            prune_step_unmasked(xi, yi, zi, A.rl2, ea, xa, 4 * s + g < n.x, lane, il, nu);
            ea = ea2;
            xa = A.xq[ea * 8 + k];
            ea2 = olu[min(4 * (s + 4) + g, n.x - 1)];
            prune_step_unmasked(xi, yi, zi, A.rl2, eb, xb, 4 * (s + 1) + g < n.x, lane, il, nu);
            eb = eb2;
            xb = A.xq[eb * 8 + k];
            eb2 = olu[min(4 * (s + 5) + g, n.x - 1)];
        }
        if (s < ns) prune_step_unmasked(xi, yi, zi, A.rl2, ea, xa, 4 * s + g < n.x, lane, il, nu);
    }
    __syncwarp();
    nb_ilist_finish(nu, nm, sd.x + ci, lane, A.cj_dummy, il, ilm, (wb ? A.seg_cnt[1] : A.seg_cnt[0]) + t);
}

// Rolling part of every segment under `nparts`, looked up by the force kernel while some part lives in inner buffer 1.
__global__ void k_seg_parts(int nseg, const int4* __restrict__ segd, int nparts, int nunits, int32_t* __restrict__ seg_part)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < nseg) seg_part[t] = nb_part_of_unit(segd[t].w, nparts, nunits);
}

// Copies the segments that live in inner buffer 1 back to buffer 0 (one warp per segment).
__global__ void k_consolidate(int nseg, const int4* __restrict__ segd, unsigned bufmask, int nparts, int nunits,
                              const int2* __restrict__ cnt1, int2* __restrict__ cnt0, const int32_t* __restrict__ il1,
                              int32_t* __restrict__ il0, const int2* __restrict__ ilm1, int2* __restrict__ ilm0)
{
    const int t = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (t >= nseg) return;
    const int4 sd = segd[t];
    if (!nb_seg_buf(sd.w, bufmask, nparts, nunits)) return;
    const int2 cnt = cnt1[t];
    for (int e = lane; e < cnt.x; e += 32) il0[sd.x + e] = il1[sd.x + e];
    for (int e = lane; e < cnt.y; e += 32) ilm0[sd.y + e] = ilm1[sd.y + e];
    if (lane == 0) cnt0[t] = cnt;
}

int launch_prune(nb_ctx* c, float rlist_inner, int part, int nparts, unsigned wmask, cudaStream_t st)
{
    const long long nu = c->nunits;
    const int u0 = (int)((long long)part * nu / nparts), u1 = (int)((long long)(part + 1) * nu / nparts);
    if (u1 <= u0) return NB_OK;
    const int32_t* order = nullptr;
    int rc = nbi_prune_order(c, nparts, &order);   // (built on the context's stream, before anything below is enqueued)
    if (rc != NB_OK) return rc;
    PruneArgs A;
    A.order = order + (size_t)u0 * 8;
    A.segd = c->segd.p;
    A.ol_cnt = c->ol_cnt.p;
    A.olu = c->olu.p;
    A.olm = c->olm.p;
    A.xq = c->xq.p;
    for (int k = 0; k < 3; k++) A.box[k] = c->box[k];
    A.rl2 = rlist_inner * rlist_inner;
    A.cj_dummy = c->nclusters_max;
    for (int b = 0; b < 2; b++) {
        A.il[b] = c->il[b].p;
        A.ilm[b] = c->ilm[b].p;
        A.seg_cnt[b] = c->seg_cnt[b].p;
    }
    A.wb = part < 32 ? (int)((wmask >> part) & 1u) : 0;   // (more than 32 parts only without the two-buffer scheme: wmask = 0)
    NB_CUDA(c, nb_launch_pdl(k_prune, dim3((u1 - u0) * 8), dim3(32), 0, st, A));
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}

// The parts of the two-buffer scheme are those of buf_nparts; a call with another nparts first moves
// every segment back to buffer 0.
int set_buf_nparts(nb_ctx* c, int nparts)
{
    if (c->buf_nparts != nparts) {
        int rc = nbi_consolidate(c);
        if (rc != NB_OK) return rc;
        c->buf_nparts = nparts;
    }
    return NB_OK;
}

// The part table the force kernel reads while some part lives in inner buffer 1: needed by the overlapped mode only.
int ensure_seg_part(nb_ctx* c)
{
    const int nparts = c->buf_nparts;
    if (c->seg_part_nparts == nparts && c->seg_part_search == c->st.search_count) return NB_OK;
    const int nseg = c->nunits * 8;
    NB_CUDA(c, c->seg_part.ensure(std::max(nseg, 1), c->stream));
    if (nseg > 0) {
        k_seg_parts<<<(nseg + 255) / 256, 256, 0, c->stream>>>(nseg, c->segd.p, nparts, c->nunits, c->seg_part.p);
        NB_LAUNCH_CHECK(c);
    }
    c->seg_part_nparts = nparts;
    c->seg_part_search = c->st.search_count;
    return NB_OK;
}

}  // namespace

// Everything a prune of `nparts` rolling parts needs besides the kernel itself (part table, launch order), built now.
int nbi_prepare_parts(nb_ctx* c, int nparts)
{
    if (nparts < 1 || nparts > 32) return NB_ERR_ARG;
    int rc = nbi_commit_pending(c);
    if (rc != NB_OK) return rc;
    if ((rc = set_buf_nparts(c, nparts)) != NB_OK) return rc;
    const int32_t* order = nullptr;
    return nbi_prune_order(c, nparts, &order);
}

int nbi_consolidate(nb_ctx* c)
{
    int rc = nbi_commit_pending(c);
    if (rc != NB_OK) return rc;
    if (c->bufmask && c->nseg_launch > 0) {
        k_consolidate<<<(c->nseg_launch * 32 + 255) / 256, 256, 0, c->stream>>>(
            c->nseg_launch, c->segd.p, c->bufmask, c->buf_nparts, c->nunits, c->seg_cnt[1].p, c->seg_cnt[0].p, c->il[1].p,
            c->il[0].p, c->ilm[1].p, c->ilm[0].p);
        NB_LAUNCH_CHECK(c);
    }
    c->bufmask = 0;
    return NB_OK;
}

// Joins an overlapped prune: the context's stream waits for it, and its part flips to the buffer it wrote.
int nbi_commit_pending(nb_ctx* c)
{
    if (c->pending_part < 0) return NB_OK;
    NB_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_side, 0));
    c->bufmask ^= 1u << c->pending_part;
    c->pending_part = -1;
    c->planes_dirty = true;
    return NB_OK;
}

int nbi_prune(nb_ctx* c, float rlist_inner, int part, int nparts)
{
    int rc = nbi_commit_pending(c);
    if (rc != NB_OK) return rc;
    if (nparts > 32 && c->bufmask) {
        if ((rc = nbi_consolidate(c)) != NB_OK) return rc;
    }
    if (c->bufmask || nparts <= 32) {
        if ((rc = set_buf_nparts(c, nparts <= 32 ? nparts : 1)) != NB_OK) return rc;
    }
    c->last_nparts = nparts;
    c->st.prune_count++;
    c->planes_dirty = true;
    NbStageTimer tm(c, NB_T_PRUNE);
    // in place: each part is rewritten in the buffer it lives in
    return launch_prune(c, rlist_inner, part, nparts, c->bufmask, c->stream);
}

int nbi_prune_overlapped(nb_ctx* c, float rlist_inner, int part, int nparts)
{
    int rc = nbi_commit_pending(c);
    if (rc != NB_OK) return rc;
    if (nparts > 32) return nb_fail(c, NB_ERR_ARG, "nb_prune_overlapped: at most 32 rolling parts (got %d)", nparts);
    cudaStream_t st = c->stream;
    if (!c->side_stream) {
        // lower priority than the caller's stream: the prune fills what the force kernel leaves free
        int lo = 0, hi = 0;
        NB_CUDA(c, cudaDeviceGetStreamPriorityRange(&lo, &hi));
        NB_CUDA(c, cudaStreamCreateWithPriority(&c->side_stream, cudaStreamNonBlocking, lo));
        NB_CUDA(c, cudaEventCreateWithFlags(&c->ev_main, cudaEventDisableTiming));
        NB_CUDA(c, cudaEventCreateWithFlags(&c->ev_side, cudaEventDisableTiming));
    }
    if (!c->have_buf1) {
        NB_CUDA(c, c->il[1].ensure(c->il[0].cap, st));
        NB_CUDA(c, c->ilm[1].ensure(c->ilm[0].cap, st));
        NB_CUDA(c, c->seg_cnt[1].ensure(c->seg_cnt[0].cap, st));
        c->have_buf1 = true;
    }
    if ((rc = set_buf_nparts(c, nparts)) != NB_OK) return rc;
    if ((rc = ensure_seg_part(c)) != NB_OK) return rc;
    c->last_nparts = nparts;
    c->st.prune_count++;
    const int32_t* order = nullptr;
    if ((rc = nbi_prune_order(c, nparts, &order)) != NB_OK) return rc;   // on the main stream, before the fork
    // fork: the side stream sees everything enqueued so far (the coordinates of the last nb_put_atoms)
    NB_CUDA(c, cudaEventRecord(c->ev_main, st));
    NB_CUDA(c, cudaStreamWaitEvent(c->side_stream, c->ev_main, 0));
    // the part is written into the buffer it does NOT live in
    const unsigned wmask = c->bufmask ^ (1u << part);
    rc = launch_prune(c, rlist_inner, part, nparts, wmask, c->side_stream);
    if (rc != NB_OK) return rc;
    NB_CUDA(c, cudaEventRecord(c->ev_side, c->side_stream));
    const long long nu = c->nunits;
    if ((int)((long long)(part + 1) * nu / nparts) > (int)((long long)part * nu / nparts)) c->pending_part = part;
    return NB_OK;
}
