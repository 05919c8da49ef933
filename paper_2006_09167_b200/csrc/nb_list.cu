// nb_list.cu -- (a3) bounding-box pair search with interaction masks, (a4) exclusion masks,
// (a5) list splitting and ordering, plus the list introspection used by the parity tests.
//
// "A joint pair list is built for the super-cluster as the union of j-clusters
// that fall in the interaction sphere of any i-cluster"; L133: "8 bits per j-cluster is
// sufficient to encode the interaction mask"; L135: "force-field exclusions are stored in the
// list with j-clusters as bitmasks"; L187: the list "is initially built using cluster
// bounding-box distances avoiding expensive all-to-all particle distance checks"; L199-L201:
// lists are sorted so long ones are not scheduled late and split when there are too few.
// The paper keeps the search on the CPU (L187); here it runs on the GPU, and so does (a5): every
// count the search produces (joint slots, work units, masks, segment extents) stays on the device
// in an NbTotals block that the next stage reads its bounds from.  Buffers are sized from the previous
// search with head-room, kernels are launched for those capacities, and the host reads the counts
// back ONCE, at the end, to learn the sizes and to check that nothing overflowed (an overflow, or the
// first search of a context, takes the "cold" path: stage by stage, sizing as it goes).
//
// Stored list: one element per (super-cluster, shift) slot "ent" = sci*14 + h (h indexes the
// zero shift and the 13 shifts s >lex 0, reading A14).  Its joint j entries occupy
// jl[ent_jbegin[ent] .. +ent_count[ent]) sorted by cj; every element starts on a multiple of
// 32 j slots so that one 32-bit word per (batch of 32 entries, i-cluster) holds one bit-plane
// of the 8-bit interaction masks.
#include "nb_internal.h"

#include <algorithm>

namespace {

// Capacities of the list buffers, passed to every stage kernel: a stage whose input count exceeds
// what the buffers hold flags the overflow and does nothing.
struct Caps {
    int jslots, units, masks, il, ilm;
};

__device__ __forceinline__ bool stage_overflow(NbTotals* t, const Caps& c)
{
    int bits = 0;
    if (t->njslots > c.jslots) bits |= NB_OVF_JOINT;
    if (t->nunits > c.units) bits |= NB_OVF_UNITS;
    if (t->nmask > c.masks) bits |= NB_OVF_MASKS;
    if (t->il_total > c.il) bits |= NB_OVF_IL;
    if (t->ilm_total > c.ilm) bits |= NB_OVF_ILM;
    bits |= t->overflow & NB_OVF_COL;   // a column did not fit its sort buffer: the layout is incomplete
    if (bits && blockIdx.x == 0 && threadIdx.x == 0) atomicOr(&t->overflow, bits);
    return bits != 0;
}

// ---------------------------------------------------------------- device scans (exclusive)
// Inputs are functors so that the flag / rounding passes need no kernel of their own.
struct FnRound32 {   // joint entries of a list element, rounded up to whole batches
    const int* cnt;
    __device__ int operator()(long long i) const { return (cnt[i] + NB_BATCH - 1) & ~(NB_BATCH - 1); }
};
struct FnArr {
    const int* a;
    __device__ int operator()(long long i) const { return a[i]; }
};
struct FnMaskFlag {   // joint entry marked by k_excl<0> (slots beyond the list are stale memory)
    const int2* jl;
    const NbTotals* tot;
    __device__ int operator()(long long i) const { return i < tot->njslots && jl[i].y != 0 ? 1 : 0; }
};

// Block-wide exclusive scan of one value per thread (1024 threads): warp shuffles + one pass over the warp sums.
__device__ __forceinline__ int block_excl_scan_1024(int v, int* s_warp /*[33]*/, int& block_total)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += u;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        int w = s_warp[lane], wi = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int u = __shfl_up_sync(0xffffffffu, wi, d);
            if (lane >= d) wi += u;
        }
        s_warp[lane] = wi - w;
        if (lane == 31) s_warp[32] = wi;
    }
    __syncthreads();
    const int out = s_warp[warp] + incl - v;
    block_total = s_warp[32];
    __syncthreads();
    return out;
}

// One block scans everything, 1024 elements at a time (for the short arrays: list elements, segments, block sums).
template <typename F>
__global__ void __launch_bounds__(1024) k_scan_1blk(F f, int* __restrict__ out, long long n, int* __restrict__ total)
{
    __shared__ int s_warp[33];
    int carry = 0;
    for (long long base = 0; base < n; base += 1024) {
        const long long i = base + threadIdx.x;
        const int v = i < n ? f(i) : 0;
        int bt;
        const int e = block_excl_scan_1024(v, s_warp, bt);
        if (i < n) out[i] = carry + e;
        carry += bt;
    }
    if (threadIdx.x == 0 && total) *total = carry;
}
template <typename F>
__global__ void __launch_bounds__(1024) k_scan_blocks(F f, int* __restrict__ out, int* __restrict__ blk, long long n)
{
    __shared__ int s_warp[33];
    const long long i = (long long)blockIdx.x * 1024 + threadIdx.x;
    const int v = i < n ? f(i) : 0;
    int bt;
    const int e = block_excl_scan_1024(v, s_warp, bt);
    if (i < n) out[i] = e;
    if (threadIdx.x == 0) blk[blockIdx.x] = bt;
}
__global__ void k_scan_add(int* __restrict__ out, const int* __restrict__ blk, long long n)
{
    long long i = (long long)blockIdx.x * 1024 + threadIdx.x;
    if (i < n) out[i] += blk[blockIdx.x];
}
// Second half of the two-launch scan: every block sums the totals of the blocks before it (a few dozen values)
// and adds that base to its 1024 outputs; the last block also writes the grand total.
__global__ void __launch_bounds__(1024) k_scan_fix(int* __restrict__ out, const int* __restrict__ blk, long long n, int nblk,
                                                   int* __restrict__ total)
{
    __shared__ int s_part[32];
    __shared__ int s_base;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int v = 0;
    for (int b = threadIdx.x; b < (int)blockIdx.x; b += 1024) v += blk[b];
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    if (lane == 0) s_part[warp] = v;
    __syncthreads();
    if (warp == 0) {
        int w = s_part[lane];
        for (int d = 16; d > 0; d >>= 1) w += __shfl_xor_sync(0xffffffffu, w, d);
        if (lane == 0) s_base = w;
    }
    __syncthreads();
    const int base = s_base;
    const long long i = (long long)blockIdx.x * 1024 + threadIdx.x;
    if (i < n) out[i] += base;
    if (total && (int)blockIdx.x == nblk - 1 && threadIdx.x == 0) *total = base + blk[nblk - 1];
}

template <typename F>
int exclusive_scan(nb_ctx* c, F f, int32_t* out, int64_t n, int32_t* total_dev)
{
    if (n <= 0) {
        if (total_dev) NB_CUDA(c, cudaMemsetAsync(total_dev, 0, sizeof(int), c->stream));
        return NB_OK;
    }
    if (n <= 4096) {   // one block, up to four rounds
        k_scan_1blk<<<1, 1024, 0, c->stream>>>(f, out, n, total_dev);
        NB_LAUNCH_CHECK(c);
        return NB_OK;
    }
    const int nblk = (int)((n + 1023) / 1024);
    NB_CUDA(c, c->scan_blk.ensure(nblk + 1, c->stream));
    k_scan_blocks<<<nblk, 1024, 0, c->stream>>>(f, out, c->scan_blk.p, n);
    NB_LAUNCH_CHECK(c);
    if (nblk <= 8192) {   // two launches: each block adds up the totals before it (a one-block scan of 21k list elements took 23 us)
        k_scan_fix<<<nblk, 1024, 0, c->stream>>>(out, c->scan_blk.p, n, nblk, total_dev);
        NB_LAUNCH_CHECK(c);
        return NB_OK;
    }
    k_scan_1blk<<<1, 1024, 0, c->stream>>>(FnArr{c->scan_blk.p}, c->scan_blk.p, nblk, total_dev);
    NB_LAUNCH_CHECK(c);
    k_scan_add<<<nblk, 1024, 0, c->stream>>>(out, c->scan_blk.p, n);
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}

// ---------------------------------------------------------------- search
struct SearchArgs {
    int nsc_max, ncx, ncy;
    int nclass;     // 2 with a local / non-local split (nb_set_local): the j side is searched per class, one list element each
    float inv_cx, inv_cy;
    float box[3];
    float rl2;      // fl32(rlist*rlist): the exact predicate's threshold (reading A12)
    float rm, rm2;  // slightly enlarged radius for the conservative candidate filters
    const int* col_sc_off;
    const float4 *sbb_lo, *sbb_hi, *bb_lo, *bb_hi;
    int* ent_count;
    const int* ent_jbegin;
    int2* jl;
    uint8_t* imask;
    NbTotals* tot;
    Caps caps;
};

// Reading A12: g_k = max(0, max(fmaf(s,L,lo_i) - hi_j, lo_j - fmaf(s,L,hi_i))), the i-side terms
// arrive pre-shifted (one fmaf each); D2 = fmaf(gz,gz, fmaf(gy,gy, gx*gx)).
__device__ __forceinline__ float bb_dist2_exact(const float* ib /*lo xyz, hi xyz (shifted)*/, float4 jlo, float4 jhi)
{
    float gx = fmaxf(fmaxf(__fsub_rn(ib[0], jhi.x), __fsub_rn(jlo.x, ib[3])), 0.f);
    float gy = fmaxf(fmaxf(__fsub_rn(ib[1], jhi.y), __fsub_rn(jlo.y, ib[4])), 0.f);
    float gz = fmaxf(fmaxf(__fsub_rn(ib[2], jhi.z), __fsub_rn(jlo.z, ib[5])), 0.f);
    return __fmaf_rn(gz, gz, __fmaf_rn(gy, gy, __fmul_rn(gx, gx)));
}

// One warp per super-cluster; lanes test 4 candidate super-clusters x 8 j-clusters at a time.
// FILL = false counts entries per (sci, shift); FILL = true repeats the enumeration and writes.
template <bool FILL>
__global__ void __launch_bounds__(128) k_search(SearchArgs A)
{
    __shared__ float s_ibb[4][8][6];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int sci = blockIdx.x * 4 + warp;
    if (sci >= A.nsc_max) return;
    if (sci >= A.tot->nsc) {   // between the actual count and the host's bound: empty list elements
        if (!FILL && lane < NB_NENT) A.ent_count[sci * NB_NENT + lane] = 0;
        return;
    }
    if (FILL && stage_overflow(A.tot, A.caps)) return;
    const int g = lane >> 3, k = lane & 7;
    const float4 ilo = A.bb_lo[sci * 8 + k], ihi = A.bb_hi[sci * 8 + k];
    const float4 slo = A.sbb_lo[sci], shi = A.sbb_hi[sci];
    if (!FILL && A.nclass == 1 && lane < NB_NHALF) A.ent_count[sci * NB_NENT + NB_NHALF + lane] = 0;   // no non-local j class
    for (int hh = 0; hh < NB_NHALF * A.nclass; hh++) {
        const int h = hh % NB_NHALF, jcls = hh / NB_NHALF;
        int sx, sy, sz;
        nb_shift_vec(nb_half_shift_id(h), sx, sy, sz);
        const float fx = (float)sx, fy = (float)sy, fz = (float)sz;
        __syncwarp();
        if (lane < 8) {
            float* b = s_ibb[warp][lane];
            b[0] = __fmaf_rn(fx, A.box[0], ilo.x);
            b[1] = __fmaf_rn(fy, A.box[1], ilo.y);
            b[2] = __fmaf_rn(fz, A.box[2], ilo.z);
            b[3] = __fmaf_rn(fx, A.box[0], ihi.x);
            b[4] = __fmaf_rn(fy, A.box[1], ihi.y);
            b[5] = __fmaf_rn(fz, A.box[2], ihi.z);
        }
        __syncwarp();
        const float tlo[3] = {__fmaf_rn(fx, A.box[0], slo.x), __fmaf_rn(fy, A.box[1], slo.y),
                              __fmaf_rn(fz, A.box[2], slo.z)};
        const float thi[3] = {__fmaf_rn(fx, A.box[0], shi.x), __fmaf_rn(fy, A.box[1], shi.y),
                              __fmaf_rn(fz, A.box[2], shi.z)};
        const int ent = sci * NB_NENT + hh;
        int count = 0;
        const int base = FILL ? A.ent_jbegin[ent] : 0;
        // candidate columns: those that can hold an atom within rm of the shifted i super-box
        const float xlo = tlo[0] - A.rm, xhi = thi[0] + A.rm, ylo = tlo[1] - A.rm, yhi = thi[1] + A.rm;
        const bool empty = xhi < 0.f || xlo > A.box[0] || yhi < 0.f || ylo > A.box[1] ||
                           thi[2] + A.rm < 0.f || tlo[2] - A.rm > A.box[2];
        if (!empty) {
            const int cx0 = max(0, (int)floorf(xlo * A.inv_cx)), cx1 = min(A.ncx - 1, (int)floorf(xhi * A.inv_cx));
            const int cy0 = max(0, (int)floorf(ylo * A.inv_cy)), cy1 = min(A.ncy - 1, (int)floorf(yhi * A.inv_cy));
            for (int cx = cx0; cx <= cx1; cx++) {
                for (int cy = cy0; cy <= cy1; cy++) {
                    const int col = cx * A.ncy + cy + jcls * A.ncx * A.ncy;
                    int s0 = A.col_sc_off[col];
                    const int s1 = A.col_sc_off[col + 1];
                    if (h == 0) s0 = max(s0, sci);   // zero shift: only cj >= ci (half list, reading A14)
                    for (int sb = s0; sb < s1; sb += 32) {
                        const int scand = sb + lane;
                        bool cand = false;
                        if (scand < s1) {
                            const float4 jlo = A.sbb_lo[scand], jhi = A.sbb_hi[scand];
                            float gx = fmaxf(fmaxf(tlo[0] - jhi.x, jlo.x - thi[0]), 0.f);
                            float gy = fmaxf(fmaxf(tlo[1] - jhi.y, jlo.y - thi[1]), 0.f);
                            float gz = fmaxf(fmaxf(tlo[2] - jhi.z, jlo.z - thi[2]), 0.f);
                            cand = gx * gx + gy * gy + gz * gz < A.rm2;
                        }
                        unsigned cmask = __ballot_sync(0xffffffffu, cand);
                        while (cmask) {
                            int p[4];
#pragma unroll
                            for (int t = 0; t < 4; t++) {
                                p[t] = cmask ? __ffs(cmask) - 1 : -1;
                                cmask &= cmask - 1;
                            }
                            const int my = g == 0 ? p[0] : (g == 1 ? p[1] : (g == 2 ? p[2] : p[3]));
                            const int scj = sb + my;
                            const int cj = scj * 8 + k;
                            unsigned imask = 0;
                            if (my >= 0) {
                                const float4 jlo = A.bb_lo[cj], jhi = A.bb_hi[cj];
#pragma unroll
                                for (int w = 0; w < 8; w++)
                                    imask |= (bb_dist2_exact(s_ibb[warp][w], jlo, jhi) < A.rl2 ? 1u : 0u) << w;
                                if (h == 0 && scj == sci) imask &= (2u << k) - 1u;   // same super-cluster: w <= k
                            }
                            const bool listed = imask != 0;
                            const unsigned lm = __ballot_sync(0xffffffffu, listed);
                            if (FILL && listed) {
                                const int pos = base + count + __popc(lm & ((1u << lane) - 1u));
                                // own super-cluster: the diagonal cluster pair needs a mask (zero shift: b > a only; under
                                // a shift, in boxes of a few cluster lengths: an atom never pairs with its own image)
                                A.jl[pos] = make_int2(cj, scj == sci ? 1 : 0);
                                A.imask[pos] = (uint8_t)imask;
                            }
                            count += __popc(lm);
                        }
                    }
                }
            }
        }
        if (!FILL && lane == 0) A.ent_count[ent] = count;
    }
}

__global__ void k_init_jl(int2* __restrict__ jl, uint8_t* __restrict__ imask, NbTotals* __restrict__ tot, Caps caps)
{
    if (stage_overflow(tot, caps)) return;
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < tot->njslots) {
        jl[i] = make_int2(-1, 0);
        imask[i] = 0;
    }
}

// One warp per batch of 32 joint entries: transpose the 32 mask bytes into 8 plane words.
__global__ void k_planes(const uint8_t* __restrict__ imask, uint32_t* __restrict__ plane, NbTotals* __restrict__ tot, Caps caps)
{
    if (stage_overflow(tot, caps)) return;
    long long b = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (b >= tot->njslots / NB_BATCH) return;
    unsigned m = imask[b * 32 + lane];
    unsigned mine = 0;
#pragma unroll
    for (int w = 0; w < 8; w++) {
        unsigned word = __ballot_sync(0xffffffffu, (m >> w) & 1u);
        if (lane == w) mine = word;
    }
    if (lane < 8) plane[b * 8 + lane] = mine;
}

// ---------------------------------------------------------------- (a5) work units, on the device
// L199-L201: "heuristically split lists to increase the available parallelism": a work unit is at most
// `ub` batches of one list element; `ub` is chosen so that there are about 6 units per SM.
__device__ __forceinline__ int unit_batches(const NbTotals* tot, int target_units)
{
    const int nbatch = tot->njslots / NB_BATCH;
    return min(NB_MAX_UNIT_BATCHES, max(1, nbatch / target_units));
}

__global__ void k_unit_count(int nent, const int* __restrict__ ent_count, const NbTotals* __restrict__ tot, int target_units,
                             int* __restrict__ nsplit)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nent) return;
    const int nb = (ent_count[e] + NB_BATCH - 1) / NB_BATCH, ub = unit_batches(tot, target_units);
    nsplit[e] = (nb + ub - 1) / ub;   // equal-sized chunks of at most ub batches
}

__global__ void k_unit_fill(int nent, const int* __restrict__ ent_count, const int* __restrict__ ent_jbegin,
                            const int* __restrict__ unit_off, NbTotals* __restrict__ tot, Caps caps, int target_units,
                            int4* __restrict__ units, int* __restrict__ batch_ent, int* __restrict__ batch_unit)
{
    if (stage_overflow(tot, caps)) return;
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nent) return;
    const int cnt = ent_count[e];
    if (!cnt) return;
    const int nb = (cnt + NB_BATCH - 1) / NB_BATCH, ub = unit_batches(tot, target_units), nsplit = (nb + ub - 1) / ub;
    const int b0 = ent_jbegin[e] / NB_BATCH, u0 = unit_off[e];
    for (int k = 0; k < nsplit; k++) {
        const int b = (int)((long long)nb * k / nsplit), bend = (int)((long long)nb * (k + 1) / nsplit);
        units[u0 + k] = make_int4(e, b0 + b, b0 + bend, e / NB_NENT);
        for (int bb = b; bb < bend; bb++) {
            batch_ent[b0 + bb] = e;
            batch_unit[b0 + bb] = u0 + k;
        }
    }
}

// ---------------------------------------------------------------- exclusion masks (a4)
struct ExclArgs {
    int natoms;
    float box[3], rl2;
    const float4 *bb_lo, *bb_hi;
    const int *excl_off, *excl_idx, *slot_of_atom, *ent_count, *ent_jbegin;
    int2* jl;
    const uint8_t* imask;
    unsigned long long* masks;
    NbTotals* tot;
    Caps caps;
};

// j class of a cluster: non-local clusters come after the local ones (nb_set_local)
__device__ __forceinline__ int cluster_class(const NbTotals* tot, int cluster) { return (cluster >> 3) >= tot->nsc_local ? 1 : 0; }

// One thread per atom; each unordered excluded pair is handled once (from its lower index; nb_init
// checks that the CSR is symmetric), in both orientations and under every shift the cluster pair is
// listed with (S:8.3.2 pairmask).  MODE 0 marks the joint entries that need a mask, MODE 1 clears the
// pair bits.  Internal bit index is b*8+a (transposed w.r.t. the ABI's a*8+b) so that the lane owning
// j-atom b reads its 8 i-atom bits as one byte.
template <int MODE>
__global__ void k_excl(ExclArgs A)
{
    if (stage_overflow(A.tot, A.caps)) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= A.natoms) return;
    for (int e = A.excl_off[i]; e < A.excl_off[i + 1]; e++) {
        int j = A.excl_idx[e];
        if (j <= i) continue;
        int sl[2] = {A.slot_of_atom[i], A.slot_of_atom[j]};
        const float4 lo[2] = {A.bb_lo[sl[0] >> 3], A.bb_lo[sl[1] >> 3]}, hi[2] = {A.bb_hi[sl[0] >> 3], A.bb_hi[sl[1] >> 3]};
#pragma unroll
        for (int o = 0; o < 2; o++) {
            int p = sl[o], q = sl[1 - o];
            int cp = p >> 3, cq = q >> 3, a = p & 7, b = q & 7;
            int scp = cp >> 3, w = cp & 7;
            for (int h = 0; h < NB_NHALF; h++) {
                // the cluster pair is listed under this shift only if its boxes pass the search's own predicate
                // (reading A13: the outer list is the pure bounding-box test): most of the 14 shifts end here,
                // without touching the list
                int sx, sy, sz;
                nb_shift_vec(nb_half_shift_id(h), sx, sy, sz);
                const float ib[6] = {__fmaf_rn((float)sx, A.box[0], lo[o].x), __fmaf_rn((float)sy, A.box[1], lo[o].y),
                                     __fmaf_rn((float)sz, A.box[2], lo[o].z), __fmaf_rn((float)sx, A.box[0], hi[o].x),
                                     __fmaf_rn((float)sy, A.box[1], hi[o].y), __fmaf_rn((float)sz, A.box[2], hi[o].z)};
                if (!(bb_dist2_exact(ib, lo[1 - o], hi[1 - o]) < A.rl2)) continue;
                int ent = scp * NB_NENT + cluster_class(A.tot, cq) * NB_NHALF + h;
                int cnt = A.ent_count[ent];
                if (cnt == 0) continue;
                int lo_ = A.ent_jbegin[ent], hi_ = lo_ + cnt;
                const int end = hi_;
                while (lo_ < hi_) {
                    int mid = (lo_ + hi_) >> 1;
                    if (A.jl[mid].x < cq) lo_ = mid + 1; else hi_ = mid;
                }
                if (lo_ < end && A.jl[lo_].x == cq && ((A.imask[lo_] >> w) & 1)) {
                    if (MODE == 0) A.jl[lo_].y = 1;
                    else atomicAnd(&A.masks[((size_t)A.jl[lo_].y * 8 + w) * 2], ~(1ull << (b * 8 + a)));
                }
            }
        }
    }
}

// Assigns mask refs (1-based; 0 = "no mask") and initialises the masks: all pairs interact,
// except on the diagonal cluster pair (cj == ci at zero shift) where only b > a is counted.
__global__ void k_excl_assign(int2* __restrict__ jl, const int* __restrict__ prefix, const int* __restrict__ batch_ent,
                              unsigned long long* __restrict__ masks, NbTotals* __restrict__ tot, Caps caps)
{
    if (stage_overflow(tot, caps)) return;
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) {
        for (int w = 0; w < 16; w++) masks[w] = ~0ull;
    }
    if (i >= tot->njslots) return;
    int2 e = jl[i];
    if (e.y == 0) return;
    int ref = prefix[i] + 1;
    jl[i].y = ref;
    int ent = batch_ent[i >> 5];
    int sci = ent / NB_NENT, h = (ent % NB_NENT) % NB_NHALF;
    unsigned long long upper = 0;   // bit b*8+a set iff b > a
    for (int b = 0; b < 8; b++)
        for (int a = 0; a < b; a++) upper |= 1ull << (b * 8 + a);
    const unsigned long long not_self = ~0x8040201008040201ull;   // bit b*8+a with b == a cleared
    for (int w = 0; w < 8; w++) {
        const bool same = e.x == sci * 8 + w, diag = h == 0 && same;
        const unsigned long long m = diag ? upper : (same ? not_self : ~0ull);   // (same cluster under a shift: all but a == b)
        masks[((size_t)ref * 8 + w) * 2] = m;       // interact
        masks[((size_t)ref * 8 + w) * 2 + 1] = m;   // counted at all
    }
}

// One warp per batch of 32 joint entries: word (batch, w) of plane_excl has bit e set iff entry e
// carries a mask whose row for i-cluster w is not all-ones (a force-field exclusion, a self pair
// or the lower triangle of a diagonal cluster pair).  The force kernel routes exactly those
// (entry, i-cluster) pairs through its masked instantiation.
__global__ void k_excl_planes(const int2* __restrict__ jl, const unsigned long long* __restrict__ masks,
                              uint32_t* __restrict__ plane_excl, NbTotals* __restrict__ tot, Caps caps)
{
    if (stage_overflow(tot, caps)) return;
    long long b = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (b >= tot->njslots / NB_BATCH) return;
    const int ref = jl[b * 32 + lane].y;
    unsigned mine = 0;
#pragma unroll
    for (int w = 0; w < 8; w++) {
        bool nt = false;
        if (ref != 0) {
            const unsigned long long* m = &masks[((size_t)ref * 8 + w) * 2];
            nt = (m[0] & m[1]) != ~0ull;
        }
        unsigned word = __ballot_sync(0xffffffffu, nt);
        if (lane == w) mine = word;
    }
    if (lane < 8) plane_excl[b * 8 + lane] = mine;
}

// ---------------------------------------------------------------- compact lists (nb_internal.h)
// Segment capacities per (work unit, i-cluster): every outer cluster pair can survive a prune.
// seg_len is the sort key of the launch orders (twice the unmasked cluster pairs, rounded up to 8, + 2 x masked pairs ~ force kernel work).
__global__ void k_ilist_caps(const int4* __restrict__ units, int nseg_cap, const uint32_t* __restrict__ plane_outer,
                             const uint32_t* __restrict__ plane_excl, NbTotals* __restrict__ tot, Caps caps,
                             int* __restrict__ capu, int* __restrict__ capm, int* __restrict__ seg_len)
{
    if (stage_overflow(tot, caps)) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nseg_cap) return;
    int nu = 0, nm = 0;
    if (i < tot->nunits * 8) {
        const int4 u = units[i >> 3];
        const int w = i & 7;
        for (int b = u.y; b < u.z; b++) {
            const unsigned bits = plane_outer[(size_t)b * 8 + w], eb = plane_excl[(size_t)b * 8 + w] & bits;
            nu += __popc(bits & ~eb);
            nm += __popc(eb);
        }
    }
    capu[i] = (8 * nu + 31) & ~31;   // j-atom entries, multiple of 32 (0 beyond the last segment: scanned as well)
    capm[i] = nm;
    seg_len[i] = min(NB_SEG_MAXKEY - 1, ((2 * nu + 7) & ~7) + 2 * nm);
}

// Counting sort of the segments, longest first inside each rolling part ("sorting to avoid long
// lists being scheduled late").  Key = part * NB_SEG_MAXKEY + (NB_SEG_MAXKEY - 1 - length); nparts = 1
// gives the force kernel's launch order.  The order among equal keys is whatever the atomics make it:
// only scheduling depends on it.
// The force kernel's order (units != nullptr, nparts = 1) is keyed by locality first (a local and a
// non-local kernel): non-empty local-local segments [0, nseg_local), longest first, then the non-empty segments that
// involve a non-local cluster [nseg_local, nseg_launch), longest first, then the empty ones.  Without nb_set_local
// every segment is local and the order is the plain longest-first one.
__device__ __forceinline__ int sort_bucket(int s0, int len, int nparts, int nunits, const int4* units, const NbTotals* tot)
{
    if (!units) return nb_part_of_unit(s0 >> 3, nparts, nunits) * NB_SEG_MAXKEY + NB_SEG_MAXKEY - 1 - len;
    if (len == 0) return 2 * NB_SEG_MAXKEY - 1;
    const int4 u = units[s0 >> 3];
    const int cls = (u.w >= tot->nsc_local || (u.x - u.w * NB_NENT) >= NB_NHALF) ? 1 : 0;
    return cls * NB_SEG_MAXKEY + NB_SEG_MAXKEY - 1 - len;
}
__global__ void k_sort_hist(const int* __restrict__ seg_len, const NbTotals* __restrict__ tot, int units_cap, int nparts,
                            const int4* __restrict__ units, int* __restrict__ hist)
{
    const int s0 = blockIdx.x * blockDim.x + threadIdx.x;
    const int nunits = tot->nunits;
    if (nunits > units_cap || s0 >= nunits * 8) return;
    atomicAdd(&hist[sort_bucket(s0, seg_len[s0], nparts, nunits, units, tot)], 1);
}
__global__ void __launch_bounds__(1024) k_sort_scan(int* __restrict__ hist, int nbuckets, NbTotals* __restrict__ tot, bool force_order)
{
    __shared__ int s_warp[33];
    int carry = 0;
    for (int base = 0; base < nbuckets; base += 1024) {
        const int i = base + threadIdx.x;
        const int v = i < nbuckets ? hist[i] : 0;
        int bt;
        const int e = block_excl_scan_1024(v, s_warp, bt);
        if (i < nbuckets) hist[i] = carry + e;
        if (force_order && i == NB_SEG_MAXKEY) tot->nseg_local = carry + e;            // everything before the non-local buckets
        if (force_order && i == 2 * NB_SEG_MAXKEY - 1) tot->nseg_launch = carry + e;   // everything before the length-0 bucket
        carry += bt;
    }
}
__global__ void k_sort_scatter(const int* __restrict__ seg_len, const NbTotals* __restrict__ tot, int units_cap, int nparts,
                               const int4* __restrict__ units, int* __restrict__ hist, int* __restrict__ seg_of_s0,
                               int* __restrict__ table)
{
    const int s0 = blockIdx.x * blockDim.x + threadIdx.x;
    const int nunits = tot->nunits;
    if (nunits > units_cap || s0 >= nunits * 8) return;
    const int pos = atomicAdd(&hist[sort_bucket(s0, seg_len[s0], nparts, nunits, units, tot)], 1);
    if (table) table[pos] = seg_of_s0[s0];   // a prune order: segment ids of each part, longest first
    else seg_of_s0[s0] = pos;                // the force kernel's order: this IS the segment id
}

struct BuildArgs {
    const int4* units;
    const uint32_t *plane, *plane_excl;
    const int2* jl;
    const int *il_off, *ilm_off, *seg_of_s0;
    int4* segd;
    int2 *ol_cnt, *seg_cnt;
    int32_t *olu, *il;
    int2 *olm, *ilm;
    int cj_dummy;
    NbTotals* tot;
    Caps caps;
};

// After a search, one block per work unit, warp w = i-cluster w: the segment's descriptor, its compact
// OUTER list (what the prune kernel streams: the cluster pairs without a mask as plain cj, those with a
// mask as {cj, mask ref}) and inner := outer (both halves of every cluster).
__global__ void __launch_bounds__(256) k_ilist_build(BuildArgs A)
{
    if (stage_overflow(A.tot, A.caps)) return;
    if (blockIdx.x >= A.tot->nunits) return;
    const int4 u = A.units[blockIdx.x];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, s0 = blockIdx.x * 8 + warp;
    const int o = A.il_off[s0], om = A.ilm_off[s0];
    const int t = A.seg_of_s0[s0];
    if (lane == 0)
        A.segd[t] = make_int4(o, om, (u.w * 8 + warp) | (nb_half_shift_id((u.x - u.w * NB_NENT) % NB_NHALF) << 26), blockIdx.x);
    const unsigned lt = (1u << lane) - 1u;
    int nu = 0, nm = 0;
    for (int b = u.y; b < u.z; b++) {
        const unsigned bits = A.plane[(size_t)b * 8 + warp], eb = A.plane_excl[(size_t)b * 8 + warp] & bits, nb = bits & ~eb;
        if ((bits >> lane) & 1u) {
            const int2 e = A.jl[(size_t)b * 32 + lane];
            if ((nb >> lane) & 1u) {
                const int p = nu + __popc(nb & lt);
                A.olu[o + p] = e.x;
                int4* dst = reinterpret_cast<int4*>(&A.il[o + 8 * p]);   // all 8 atoms of the j-cluster
                dst[0] = make_int4(8 * e.x, 8 * e.x + 1, 8 * e.x + 2, 8 * e.x + 3);
                dst[1] = make_int4(8 * e.x + 4, 8 * e.x + 5, 8 * e.x + 6, 8 * e.x + 7);
            } else {
                const int p = nm + __popc(eb & lt);
                A.olm[om + p] = e;
                A.ilm[om + p] = e;
            }
        }
        nu += __popc(nb);
        nm += __popc(eb);
    }
    if (lane == 0) A.ol_cnt[t] = make_int2(nu, nm);
    __syncwarp();
    nb_ilist_finish(8 * nu, nm, u.y * 8 + warp, lane, A.cj_dummy, A.il + o, A.ilm + om, &A.seg_cnt[t]);
}

// ---------------------------------------------------------------- introspection
__global__ void k_count_bits(const uint32_t* __restrict__ plane, long long nwords, long long* __restrict__ out)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int c = i < nwords ? __popc(plane[i]) : 0;
    for (int d = 16; d > 0; d >>= 1) c += __shfl_xor_sync(0xffffffffu, c, d);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd((unsigned long long*)out, (unsigned long long)c);
}

__global__ void k_count_joint(const uint8_t* __restrict__ imask, const int2* __restrict__ jl, long long n,
                              long long* __restrict__ out /* [0]=joint entries, [1]=masked */)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int a = i < n && imask[i] ? 1 : 0, m = i < n && jl[i].y != 0 ? 1 : 0;
    for (int d = 16; d > 0; d >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, d);
        m += __shfl_xor_sync(0xffffffffu, m, d);
    }
    if ((threadIdx.x & 31) == 0) {
        if (a) atomicAdd((unsigned long long*)&out[0], (unsigned long long)a);
        if (m) atomicAdd((unsigned long long*)&out[1], (unsigned long long)m);
    }
}

__global__ void k_count_nonempty(const int* __restrict__ ent_count, int nent, long long* __restrict__ out)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int a = i < nent && ent_count[i] > 0 ? 1 : 0;
    for (int d = 16; d > 0; d >>= 1) a += __shfl_xor_sync(0xffffffffu, a, d);
    if ((threadIdx.x & 31) == 0 && a) atomicAdd((unsigned long long*)out, (unsigned long long)a);
}

// plane_inner (the inner list at cluster-pair granularity, which only the dumps and the pair counting
// read) from the compact inner list the force kernel streams: one warp per segment; a listed j atom or
// masked cluster pair sets the bit of its joint entry, found by bisection in the unit's slice of jl.
__global__ void k_planes_from_il(int nseg, const int4* __restrict__ segd, const int2* __restrict__ cnt0, const int2* __restrict__ cnt1,
                                 const int32_t* __restrict__ il0, const int32_t* __restrict__ il1, const int2* __restrict__ ilm0,
                                 const int2* __restrict__ ilm1, const int4* __restrict__ units, const int* __restrict__ ent_count,
                                 const int* __restrict__ ent_jbegin, const int2* __restrict__ jl, unsigned bufmask, int nparts,
                                 int nunits, int nslot_real, uint32_t* __restrict__ plane_inner)
{
    const int t = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (t >= nseg) return;
    const int4 sd = segd[t];
    const int buf = nb_seg_buf(sd.w, bufmask, nparts, nunits);
    const int2 cnt = buf ? cnt1[t] : cnt0[t];
    const int32_t* il = (buf ? il1 : il0) + sd.x;
    const int2* ilm = (buf ? ilm1 : ilm0) + sd.y;
    const int4 u = units[sd.w];
    const int w = sd.z & 7;
    const int jb = u.y * NB_BATCH, je = min(u.z * NB_BATCH, ent_jbegin[u.x] + ent_count[u.x]);
    for (int e = lane; e < cnt.x + cnt.y; e += 32) {
        int cj;
        if (e < cnt.x) {
            const int slot = il[e];
            if (slot >= nslot_real) continue;   // dummy padding
            cj = slot >> 3;
        } else {
            cj = ilm[e - cnt.x].x;
        }
        int lo = jb, hi = je;
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (jl[mid].x < cj) lo = mid + 1; else hi = mid;
        }
        atomicOr(&plane_inner[(size_t)(lo >> 5) * 8 + w], 1u << (lo & 31));
    }
}

__device__ __forceinline__ unsigned entry_bits(const uint32_t* plane, long long e)
{
    unsigned bits = 0;
    const uint32_t* p = plane + (e >> 5) * 8;
#pragma unroll
    for (int w = 0; w < 8; w++) bits |= ((p[w] >> (e & 31)) & 1u) << w;
    return bits;
}

struct FnEntryBits {
    const uint32_t* plane;
    __device__ int operator()(long long e) const { return __popc(entry_bits(plane, e)); }
};

struct DumpArgs {
    const uint32_t* plane;
    const int* offset;
    const int2* jl;
    const int *batch_ent, *batch_unit, *atom_of_slot;
    const unsigned long long* masks;
    long long n;
    int nunits, nparts;
    int32_t *ci, *cj, *shift, *part;
    uint64_t* pairmask;
};

__global__ void k_dump_fill(DumpArgs A)
{
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= A.n) return;
    unsigned bits = entry_bits(A.plane, e);
    if (!bits) return;
    int2 je = A.jl[e];
    int ent = A.batch_ent[e >> 5];
    int sci = ent / NB_NENT, h = (ent % NB_NENT) % NB_NHALF;
    const int part = nb_part_of_unit(A.batch_unit[e >> 5], A.nparts, A.nunits);
    unsigned jvalid = 0;
    for (int b = 0; b < 8; b++) jvalid |= (A.atom_of_slot[je.x * 8 + b] >= 0 ? 1u : 0u) << b;
    int o = A.offset[e];
    for (int w = 0; w < 8; w++) {
        if (!((bits >> w) & 1)) continue;
        int ci = sci * 8 + w;
        if (A.ci) A.ci[o] = ci;
        if (A.cj) A.cj[o] = je.x;
        if (A.shift) A.shift[o] = nb_half_shift_id(h);
        if (A.part) A.part[o] = part;
        if (A.pairmask) {
            unsigned long long mi = A.masks[((size_t)je.y * 8 + w) * 2];       // interact, bit b*8+a
            mi &= A.masks[((size_t)je.y * 8 + w) * 2 + 1];                    // and counted
            unsigned long long out = 0;
            for (int a = 0; a < 8; a++) {
                if (A.atom_of_slot[ci * 8 + a] < 0) continue;
                for (int b = 0; b < 8; b++)
                    if (((jvalid >> b) & 1) && ((mi >> (b * 8 + a)) & 1)) out |= 1ull << (a * 8 + b);
            }
            A.pairmask[o] = out;
        }
        o++;
    }
}

// ---------------------------------------------------------------- buffer sizing
size_t with_headroom(size_t n, size_t floor_) { return std::max(floor_, n + n / 4 + 64); }

int size_joint(nb_ctx* c, size_t njslots)
{
    if (njslots <= c->cap_jslots && c->cap_jslots > 0) return NB_OK;
    cudaStream_t st = c->stream;
    const size_t cap = (with_headroom(njslots, 4096) + NB_BATCH - 1) / NB_BATCH * NB_BATCH;
    NB_CUDA(c, c->jl.ensure(cap, st));
    NB_CUDA(c, c->imask_outer.ensure(cap, st));
    NB_CUDA(c, c->plane_outer.ensure(cap / NB_BATCH * 8, st));
    NB_CUDA(c, c->plane_inner.ensure(cap / NB_BATCH * 8, st));
    NB_CUDA(c, c->plane_excl.ensure(cap / NB_BATCH * 8, st));
    NB_CUDA(c, c->batch_ent.ensure(cap / NB_BATCH * 2, st));
    c->cap_jslots = cap;
    return NB_OK;
}
int size_units(nb_ctx* c, size_t nunits)
{
    if (nunits <= c->cap_units && c->cap_units > 0) return NB_OK;
    cudaStream_t st = c->stream;
    const size_t cap = with_headroom(nunits, 256), nseg = cap * 8;
    NB_CUDA(c, c->units_canon.ensure(cap, st));
    NB_CUDA(c, c->il_off.ensure(nseg, st));
    NB_CUDA(c, c->ilm_off.ensure(nseg, st));
    NB_CUDA(c, c->seg_of_s0.ensure(nseg, st));
    NB_CUDA(c, c->segd.ensure(nseg, st));
    NB_CUDA(c, c->ol_cnt.ensure(nseg, st));
    NB_CUDA(c, c->seg_cnt[0].ensure(nseg, st));
    if (c->have_buf1) NB_CUDA(c, c->seg_cnt[1].ensure(nseg, st));
    c->cap_units = cap;
    return NB_OK;
}
int size_masks(nb_ctx* c, size_t nmask)
{
    if (nmask <= c->cap_masks && c->cap_masks > 0) return NB_OK;
    const size_t cap = with_headroom(nmask, 256);
    NB_CUDA(c, c->excl_masks.ensure((cap + 1) * 16, c->stream));
    c->cap_masks = cap;
    return NB_OK;
}
int size_il(nb_ctx* c, size_t il_total, size_t ilm_total)
{
    cudaStream_t st = c->stream;
    if (il_total > c->cap_il || c->cap_il == 0) {
        const size_t cap = with_headroom(il_total, 4096);
        NB_CUDA(c, c->il[0].ensure(cap + 8, st));
        NB_CUDA(c, c->olu.ensure(cap + 8, st));
        if (c->have_buf1) NB_CUDA(c, c->il[1].ensure(cap + 8, st));
        c->cap_il = cap;
    }
    if (ilm_total > c->cap_ilm || c->cap_ilm == 0) {
        const size_t cap = with_headroom(ilm_total, 1024);
        NB_CUDA(c, c->ilm[0].ensure(cap + 8, st));
        NB_CUDA(c, c->olm.ensure(cap + 8, st));
        if (c->have_buf1) NB_CUDA(c, c->ilm[1].ensure(cap + 8, st));
        c->cap_ilm = cap;
    }
    return NB_OK;
}

int read_totals(nb_ctx* c)
{
    NB_CUDA(c, cudaMemcpyAsync(c->tot_host, c->tot_dev, sizeof(NbTotals), cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    return NB_OK;
}

const int NB_RETRY = 1;

int sort_segments(nb_ctx* c, int nparts, int nseg_cap, const int* seg_len, int* table)
{
    cudaStream_t st = c->stream;
    const bool force_order = table == nullptr;   // (then nparts = 1): keyed by locality, then length
    const int4* units = force_order ? c->units_canon.p : nullptr;
    const int nbuckets = force_order ? 2 * NB_SEG_MAXKEY : nparts * NB_SEG_MAXKEY;
    NB_CUDA(c, c->sort_hist.ensure(nbuckets, st));
    NB_CUDA(c, cudaMemsetAsync(c->sort_hist.p, 0, sizeof(int) * nbuckets, st));
    k_sort_hist<<<(nseg_cap + 255) / 256, 256, 0, st>>>(seg_len, c->tot_dev, (int)c->cap_units, nparts, units, c->sort_hist.p);
    NB_LAUNCH_CHECK(c);
    k_sort_scan<<<1, 1024, 0, st>>>(c->sort_hist.p, nbuckets, c->tot_dev, force_order);
    NB_LAUNCH_CHECK(c);
    k_sort_scatter<<<(nseg_cap + 255) / 256, 256, 0, st>>>(seg_len, c->tot_dev, (int)c->cap_units, nparts, units, c->sort_hist.p,
                                                           c->seg_of_s0.p, table);
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}

// One pass over (a2)-(a5).  Returns NB_RETRY when a buffer sized from the previous search was too small
// (the context is then "cold": the next attempt sizes as it goes).
int search_attempt(nb_ctx* c, float rlist)
{
    cudaStream_t st = c->stream;
    const bool cold = c->cold;
    NB_CUDA(c, cudaMemsetAsync(c->tot_dev, 0, sizeof(NbTotals), st));
    int rc = nbi_grid(c);
    if (rc != NB_OK) return rc;
    NbStageTimer* tm = new NbStageTimer(c, NB_T_SEARCH);
    struct TmGuard { NbStageTimer*& t; ~TmGuard() { delete t; } } tm_guard{tm};
    const int nsc_max = c->nsc_max;
    c->nent = nsc_max * NB_NENT;
    const int nent = c->nent;
    NB_CUDA(c, c->ent_count.ensure(nent + 1, st));
    NB_CUDA(c, c->ent_jbegin.ensure(nent + 1, st));
    NB_CUDA(c, c->unit_nsplit.ensure(nent + 1, st));
    NB_CUDA(c, c->unit_off.ensure(nent + 1, st));
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, c->prm.device);
    const int target_units = 6 * nsm;   // about 6 prune work units per SM (measured best on configs 1-3)

    SearchArgs A;
    A.nclass = c->nclass;
    A.nsc_max = nsc_max; A.ncx = c->ncx; A.ncy = c->ncy; A.inv_cx = c->inv_cx; A.inv_cy = c->inv_cy;
    for (int k = 0; k < 3; k++) A.box[k] = c->box[k];
    A.rl2 = rlist * rlist;
    A.rm = rlist * (1.0f + 1e-5f) + 1e-5f;
    A.rm2 = A.rm * A.rm;
    A.col_sc_off = c->col_sc_off.p;
    A.sbb_lo = c->sbb_lo.p; A.sbb_hi = c->sbb_hi.p; A.bb_lo = c->bb_lo.p; A.bb_hi = c->bb_hi.p;
    A.ent_count = c->ent_count.p; A.ent_jbegin = nullptr; A.jl = nullptr; A.imask = nullptr;
    A.tot = c->tot_dev;
    A.caps = Caps{0, 0, 0, 0, 0};
    k_search<false><<<(nsc_max + 3) / 4, 128, 0, st>>>(A);
    NB_LAUNCH_CHECK(c);
    // element offsets (32-aligned) and the number of joint slots
    rc = exclusive_scan(c, FnRound32{c->ent_count.p}, c->ent_jbegin.p, nent, &c->tot_dev->njslots);
    if (rc != NB_OK) return rc;
    if (cold) {
        if ((rc = read_totals(c)) != NB_OK) return rc;
        if ((long long)c->tot_host->njslots > 0x7fffff00LL || c->tot_host->njslots < 0)
            return nb_fail(c, NB_ERR_OVERFLOW, "pair list exceeds 2^31 joint entries");
        if ((rc = size_joint(c, c->tot_host->njslots)) != NB_OK) return rc;
    }
    // (a5) split into bounded work units
    k_unit_count<<<(nent + 255) / 256, 256, 0, st>>>(nent, c->ent_count.p, c->tot_dev, target_units, c->unit_nsplit.p);
    NB_LAUNCH_CHECK(c);
    rc = exclusive_scan(c, FnArr{c->unit_nsplit.p}, c->unit_off.p, nent, &c->tot_dev->nunits);
    if (rc != NB_OK) return rc;
    if (cold) {
        if ((rc = read_totals(c)) != NB_OK) return rc;
        if ((rc = size_units(c, c->tot_host->nunits)) != NB_OK) return rc;
        if ((rc = size_masks(c, c->cap_masks)) != NB_OK) return rc;
        if ((rc = size_il(c, c->cap_il, c->cap_ilm)) != NB_OK) return rc;
    }
    NB_CUDA(c, c->scan_tmp.ensure(std::max(c->cap_jslots * 2, c->cap_units * 8 * 3) + 64, st));
    Caps caps{(int)c->cap_jslots, (int)c->cap_units, (int)c->cap_masks, (int)c->cap_il, (int)c->cap_ilm};
    if (cold) caps.masks = caps.il = caps.ilm = 0x7fffffff;   // sized below, before anything is written
    A.caps = caps;
    int* d_batch_unit = c->batch_ent.p + c->cap_jslots / NB_BATCH;
    k_unit_fill<<<(nent + 255) / 256, 256, 0, st>>>(nent, c->ent_count.p, c->ent_jbegin.p, c->unit_off.p, c->tot_dev, caps,
                                                    target_units, c->units_canon.p, c->batch_ent.p, d_batch_unit);
    NB_LAUNCH_CHECK(c);
    const unsigned gj = (unsigned)((c->cap_jslots + 255) / 256), gb = (unsigned)((c->cap_jslots + 255) / 256);
    k_init_jl<<<gj, 256, 0, st>>>(c->jl.p, c->imask_outer.p, c->tot_dev, caps);
    NB_LAUNCH_CHECK(c);
    A.ent_jbegin = c->ent_jbegin.p; A.jl = c->jl.p; A.imask = c->imask_outer.p;
    k_search<true><<<(nsc_max + 3) / 4, 128, 0, st>>>(A);
    NB_LAUNCH_CHECK(c);
    k_planes<<<gb, 256, 0, st>>>(c->imask_outer.p, c->plane_outer.p, c->tot_dev, caps);
    NB_LAUNCH_CHECK(c);

    // (a4) exclusion masks
    delete tm;
    tm = new NbStageTimer(c, NB_T_MASKS);
    ExclArgs E;
    E.natoms = c->natoms;
    for (int k = 0; k < 3; k++) E.box[k] = c->box[k];
    E.rl2 = rlist * rlist;
    E.bb_lo = c->bb_lo.p; E.bb_hi = c->bb_hi.p;
    E.excl_off = c->excl_off.p; E.excl_idx = c->excl_idx.p; E.slot_of_atom = c->slot_of_atom.p;
    E.ent_count = c->ent_count.p; E.ent_jbegin = c->ent_jbegin.p; E.jl = c->jl.p; E.imask = c->imask_outer.p;
    E.masks = nullptr; E.tot = c->tot_dev; E.caps = caps;
    if (c->nexcl) {
        k_excl<0><<<(c->natoms + 127) / 128, 128, 0, st>>>(E);
        NB_LAUNCH_CHECK(c);
    }
    int* prefix = c->scan_tmp.p;
    rc = exclusive_scan(c, FnMaskFlag{c->jl.p, c->tot_dev}, prefix, (int64_t)c->cap_jslots, &c->tot_dev->nmask);
    if (rc != NB_OK) return rc;
    if (cold) {
        if ((rc = read_totals(c)) != NB_OK) return rc;
        if ((rc = size_masks(c, c->tot_host->nmask)) != NB_OK) return rc;
        caps.masks = (int)c->cap_masks;
    }
    k_excl_assign<<<gj, 256, 0, st>>>(c->jl.p, prefix, c->batch_ent.p, c->excl_masks.p, c->tot_dev, caps);
    NB_LAUNCH_CHECK(c);
    if (c->nexcl) {
        E.masks = c->excl_masks.p; E.caps = caps;
        k_excl<1><<<(c->natoms + 127) / 128, 128, 0, st>>>(E);
        NB_LAUNCH_CHECK(c);
    }
    k_excl_planes<<<gb, 256, 0, st>>>(c->jl.p, c->excl_masks.p, c->plane_excl.p, c->tot_dev, caps);
    NB_LAUNCH_CHECK(c);

    // compact lists: segment capacities from the outer counts, offsets, launch order, then inner := outer
    const int nseg_cap = (int)c->cap_units * 8;
    int* capu = c->scan_tmp.p;
    int* capm = capu + nseg_cap;
    int* seg_len = capm + nseg_cap;
    k_ilist_caps<<<(nseg_cap + 255) / 256, 256, 0, st>>>(c->units_canon.p, nseg_cap, c->plane_outer.p, c->plane_excl.p, c->tot_dev,
                                                        caps, capu, capm, seg_len);
    NB_LAUNCH_CHECK(c);
    rc = exclusive_scan(c, FnArr{capu}, c->il_off.p, nseg_cap, &c->tot_dev->il_total);
    if (rc != NB_OK) return rc;
    rc = exclusive_scan(c, FnArr{capm}, c->ilm_off.p, nseg_cap, &c->tot_dev->ilm_total);
    if (rc != NB_OK) return rc;
    if (cold) {
        if ((rc = read_totals(c)) != NB_OK) return rc;
        if ((rc = size_il(c, c->tot_host->il_total, c->tot_host->ilm_total)) != NB_OK) return rc;
        caps.il = (int)c->cap_il;
        caps.ilm = (int)c->cap_ilm;
    }
    if ((rc = sort_segments(c, 1, nseg_cap, seg_len, nullptr)) != NB_OK) return rc;
    BuildArgs B;
    B.units = c->units_canon.p; B.plane = c->plane_outer.p; B.plane_excl = c->plane_excl.p; B.jl = c->jl.p;
    B.il_off = c->il_off.p; B.ilm_off = c->ilm_off.p; B.seg_of_s0 = c->seg_of_s0.p; B.segd = c->segd.p;
    B.ol_cnt = c->ol_cnt.p; B.seg_cnt = c->seg_cnt[0].p; B.olu = c->olu.p; B.il = c->il[0].p; B.olm = c->olm.p;
    B.ilm = c->ilm[0].p; B.cj_dummy = c->nclusters_max; B.tot = c->tot_dev; B.caps = caps;
    k_ilist_build<<<(unsigned)c->cap_units, 256, 0, st>>>(B);
    NB_LAUNCH_CHECK(c);
    // segment lengths are kept for the prune orders (scan_tmp is reused by the dumps)
    NB_CUDA(c, c->seg_len.ensure(nseg_cap, st));
    NB_CUDA(c, cudaMemcpyAsync(c->seg_len.p, seg_len, sizeof(int) * nseg_cap, cudaMemcpyDeviceToDevice, st));
    if ((rc = nbi_ljrows(c)) != NB_OK) return rc;

    // the one synchronisation of a warm search: the counts, and whether everything fitted
    if ((rc = read_totals(c)) != NB_OK) return rc;
    const NbTotals& T = *c->tot_host;
    if (T.bad_type) return nb_fail(c, NB_ERR_ARG, "an atom type is outside [0, %d)", c->ntypes);
    if (T.overflow) {
        if (cold) return nb_fail(c, NB_ERR_OVERFLOW, "list buffers overflowed on the sizing pass (flags %d)", T.overflow);
        c->cold = true;
        return NB_RETRY;
    }
    c->cold = false;
    c->nsc = T.nsc;
    c->max_col_count = T.max_col;
    c->nclusters = c->nsc * NB_SUPER_SIZE;
    c->nslots = c->nsc * NB_SC_ATOMS;
    c->njslots = T.njslots;
    c->nbatch = T.njslots / NB_BATCH;
    c->nunits = T.nunits;
    c->nmask = T.nmask;
    c->il_total = T.il_total;
    c->ilm_total = T.ilm_total;
    c->nseg_launch = T.nseg_launch;
    c->nseg_local = T.nseg_local;
    c->nsc_local = T.nsc_local;
    c->st.nsuper = c->nsc;
    c->st.nclusters = c->nclusters;
    c->st.nslots = c->nslots;
    return NB_OK;
}

}  // namespace

int nbi_exclusive_scan(nb_ctx* c, const int32_t* in, int32_t* out, int64_t n, int32_t* total_dev)
{
    return exclusive_scan(c, FnArr{in}, out, n, total_dev);
}

static int count_bits(nb_ctx* c, const uint32_t* plane, int64_t* out)
{
    NB_CUDA(c, c->counters.ensure(8, c->stream));
    NB_CUDA(c, cudaMemsetAsync(c->counters.p, 0, 8 * sizeof(long long), c->stream));
    long long nwords = c->nbatch * 8;
    if (nwords) {
        k_count_bits<<<(unsigned)((nwords + 255) / 256), 256, 0, c->stream>>>(plane, nwords, c->counters.p);
        NB_LAUNCH_CHECK(c);
    }
    long long v = 0;
    NB_CUDA(c, cudaMemcpyAsync(&v, c->counters.p, sizeof(v), cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    *out = v;
    return NB_OK;
}

int nbi_rebuild_inner_planes(nb_ctx* c)
{
    if (!c->planes_dirty) return NB_OK;
    int rc = nbi_commit_pending(c);
    if (rc != NB_OK) return rc;
    cudaStream_t st = c->stream;
    if (c->nbatch) NB_CUDA(c, cudaMemsetAsync(c->plane_inner.p, 0, sizeof(uint32_t) * c->nbatch * 8, st));
    if (c->nseg_launch > 0) {
        k_planes_from_il<<<(c->nseg_launch * 32 + 255) / 256, 256, 0, st>>>(
            c->nseg_launch, c->segd.p, c->seg_cnt[0].p, c->seg_cnt[1].p, c->il[0].p, c->il[1].p, c->ilm[0].p, c->ilm[1].p,
            c->units_canon.p, c->ent_count.p, c->ent_jbegin.p, c->jl.p, c->bufmask, c->buf_nparts, c->nunits,
            8 * c->nclusters_max, c->plane_inner.p);
        NB_LAUNCH_CHECK(c);
    }
    c->planes_dirty = false;
    return NB_OK;
}

int nbi_list_count(nb_ctx* c, int which, int64_t* n)
{
    if (which == 1) {
        int rc = nbi_rebuild_inner_planes(c);
        if (rc != NB_OK) return rc;
    }
    return count_bits(c, which == 0 ? c->plane_outer.p : c->plane_inner.p, n);
}

// List statistics of nb_stats, computed when asked for (nb_get_stats), not in every search.
int nbi_list_stats(nb_ctx* c)
{
    if (!c->stats_dirty) return NB_OK;
    cudaStream_t st = c->stream;
    NB_CUDA(c, c->counters.ensure(8, st));
    NB_CUDA(c, cudaMemsetAsync(c->counters.p, 0, 8 * sizeof(long long), st));
    if (c->nbatch) {
        k_count_bits<<<(unsigned)((c->nbatch * 8 + 255) / 256), 256, 0, st>>>(c->plane_outer.p, c->nbatch * 8, c->counters.p);
        NB_LAUNCH_CHECK(c);
        k_count_joint<<<(unsigned)((c->njslots + 255) / 256), 256, 0, st>>>(c->imask_outer.p, c->jl.p, c->njslots, c->counters.p + 1);
        NB_LAUNCH_CHECK(c);
    }
    k_count_nonempty<<<(c->nent + 255) / 256, 256, 0, st>>>(c->ent_count.p, c->nent, c->counters.p + 3);
    NB_LAUNCH_CHECK(c);
    long long cnt[4] = {0, 0, 0, 0};
    NB_CUDA(c, cudaMemcpyAsync(cnt, c->counters.p, sizeof(cnt), cudaMemcpyDeviceToHost, st));
    NB_CUDA(c, cudaStreamSynchronize(st));
    c->st.n_pairs_outer = cnt[0];
    c->st.n_joint_outer = cnt[1];
    c->st.n_excl_masks = cnt[2];
    c->st.n_sci_entries = cnt[3];
    c->st.n_work_units = c->nunits;
    c->stats_dirty = false;
    return NB_OK;
}

int nbi_search(nb_ctx* c, float rlist)
{
    int rc = nbi_commit_pending(c);
    if (rc != NB_OK) return rc;
    c->bufmask = 0;
    c->buf_nparts = 1;
    for (int attempt = 0; attempt < 3; attempt++) {
        rc = search_attempt(c, rlist);
        if (rc != NB_RETRY) break;
        c->st.list_grow_retries++;
    }
    if (rc == NB_RETRY) return nb_fail(c, NB_ERR_OVERFLOW, "list buffers kept overflowing");
    if (rc != NB_OK) {
        c->cold = true;
        return rc;
    }
    c->rlist_outer = rlist;
    c->last_nparts = 1;
    c->have_list = true;
    c->stats_dirty = true;
    c->planes_dirty = true;
    c->st.search_count++;
    return NB_OK;
}

// Launch order of the prune kernel for rolling parts of `nparts`: segment ids, part by part (part p
// occupies [8*u0(p), 8*u1(p)) of the table), longest outer list first inside each part.  Built on the
// device once per (search, nparts).
int nbi_prune_order(nb_ctx* c, int nparts, const int32_t** table)
{
    nb_ctx::PruneOrder* po = nullptr;
    for (auto& e : c->prune_orders)
        if (e.nparts == nparts && e.search == c->st.search_count) po = &e;
    if (!po) {
        po = &c->prune_orders[c->prune_order_next];
        c->prune_order_next = (c->prune_order_next + 1) % 4;
        const int nseg = c->nunits * 8;
        NB_CUDA(c, po->d.ensure(std::max(nseg, 1), c->stream));
        // more parts than the sort has buckets for: one part per key range is pointless, keep canonical order
        const int sort_parts = nparts <= NB_MAX_SORT_PARTS ? nparts : 1;
        if (nseg > 0) {
            if (sort_parts == nparts) {
                int rc = sort_segments(c, nparts, nseg, c->seg_len.p, po->d.p);
                if (rc != NB_OK) return rc;
            } else {
                NB_CUDA(c, cudaMemcpyAsync(po->d.p, c->seg_of_s0.p, sizeof(int) * nseg, cudaMemcpyDeviceToDevice, c->stream));
            }
        }
        po->nparts = nparts;
        po->search = c->st.search_count;
    }
    *table = po->d.p;
    return NB_OK;
}

int nbi_list_dump(nb_ctx* c, int which, int32_t* ci, int32_t* cj, int32_t* shift, uint64_t* pairmask, int32_t* part)
{
    if (!c->nbatch) return NB_OK;
    cudaStream_t st = c->stream;
    if (which == 1) {
        int rc = nbi_rebuild_inner_planes(c);
        if (rc != NB_OK) return rc;
    }
    const uint32_t* plane = which == 0 ? c->plane_outer.p : c->plane_inner.p;
    int* off = c->scan_tmp.p;
    int rc = exclusive_scan(c, FnEntryBits{plane}, off, c->njslots, nullptr);
    if (rc != NB_OK) return rc;
    DumpArgs D;
    D.plane = plane; D.offset = off; D.jl = c->jl.p; D.batch_ent = c->batch_ent.p;
    D.batch_unit = c->batch_ent.p + c->cap_jslots / NB_BATCH;
    D.atom_of_slot = c->atom_of_slot.p; D.masks = c->excl_masks.p; D.n = c->njslots;
    D.nunits = std::max(c->nunits, 1); D.nparts = std::max(c->last_nparts, 1);
    D.ci = ci; D.cj = cj; D.shift = shift; D.part = part; D.pairmask = pairmask;
    k_dump_fill<<<(unsigned)((c->njslots + 255) / 256), 256, 0, st>>>(D);
    NB_LAUNCH_CHECK(c);
    NB_CUDA(c, cudaStreamSynchronize(st));
    return NB_OK;
}
