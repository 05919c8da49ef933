// nb_list.cu -- (a3) bounding-box pair search with interaction masks, (a4) exclusion masks,
// (a5) list splitting and ordering, plus the list introspection used by the parity tests.
//
// "A joint pair list is built for the super-cluster as the union of j-clusters
// that fall in the interaction sphere of any i-cluster"; L133: "8 bits per j-cluster is
// sufficient to encode the interaction mask"; L135: "force-field exclusions are stored in the
// list with j-clusters as bitmasks"; L187: the list "is initially built using cluster
// bounding-box distances avoiding expensive all-to-all particle distance checks"; L199-L201:
// lists are sorted so long ones are not scheduled late and split when there are too few.
// The paper keeps the search on the CPU (L187); here it runs on the GPU.
//
// Stored list: one element per (super-cluster, shift) slot "ent" = sci*14 + h (h indexes the
// zero shift and the 13 shifts s >lex 0, reading A14).  Its joint j entries occupy
// jl[ent_jbegin[ent] .. +ent_count[ent]) sorted by cj; every element starts on a multiple of
// 32 j slots so that one 32-bit word per (batch of 32 entries, i-cluster) holds one bit-plane
// of the 8-bit interaction masks: warp w of a block gets "which of these 32 j-clusters
// interact with i-cluster w" with a single load instead of a ballot over 32 bytes.
#include "nb_internal.h"

#include <algorithm>

namespace {

// ---------------------------------------------------------------- device scan (exclusive)
__global__ void k_scan1(const int* __restrict__ in, int* __restrict__ out, int* __restrict__ blk, long long n)
{
    __shared__ int s[1024];
    long long i = (long long)blockIdx.x * 1024 + threadIdx.x;
    int t = threadIdx.x;
    int v = i < n ? in[i] : 0;
    s[t] = v;
    __syncthreads();
    for (int d = 1; d < 1024; d <<= 1) {
        int u = t >= d ? s[t - d] : 0;
        __syncthreads();
        s[t] += u;
        __syncthreads();
    }
    if (i < n) out[i] = s[t] - v;
    if (t == 1023) blk[blockIdx.x] = s[t];
}
__global__ void k_scan2(int* __restrict__ blk, int nblk, int* __restrict__ total)
{
    __shared__ int s[1024];
    __shared__ int carry;
    int t = threadIdx.x;
    if (t == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < nblk; base += 1024) {
        int v = base + t < nblk ? blk[base + t] : 0;
        s[t] = v;
        __syncthreads();
        for (int d = 1; d < 1024; d <<= 1) {
            int u = t >= d ? s[t - d] : 0;
            __syncthreads();
            s[t] += u;
            __syncthreads();
        }
        if (base + t < nblk) blk[base + t] = carry + s[t] - v;
        __syncthreads();
        if (t == 1023) carry += s[t];
        __syncthreads();
    }
    if (t == 0 && total) *total = carry;
}
__global__ void k_scan3(int* __restrict__ out, const int* __restrict__ blk, long long n)
{
    long long i = (long long)blockIdx.x * 1024 + threadIdx.x;
    if (i < n) out[i] += blk[blockIdx.x];
}

// ---------------------------------------------------------------- search
struct SearchArgs {
    int nsc, ncx, ncy;
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
    if (sci >= A.nsc) return;
    const int g = lane >> 3, k = lane & 7;
    const float4 ilo = A.bb_lo[sci * 8 + k], ihi = A.bb_hi[sci * 8 + k];
    const float4 slo = A.sbb_lo[sci], shi = A.sbb_hi[sci];
    for (int h = 0; h < NB_NHALF; h++) {
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
        const int ent = sci * NB_NHALF + h;
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
                    const int col = cx * A.ncy + cy;
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
                                A.jl[pos] = make_int2(cj, (h == 0 && scj == sci) ? 1 : 0);
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

__global__ void k_init_jl(int2* __restrict__ jl, long long n)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) jl[i] = make_int2(-1, 0);
}

// One warp per batch of 32 joint entries: transpose the 32 mask bytes into 8 plane words.
__global__ void k_planes(const uint8_t* __restrict__ imask, uint32_t* __restrict__ plane, long long nbatch)
{
    long long b = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (b >= nbatch) return;
    unsigned m = imask[b * 32 + lane];
    unsigned mine = 0;
#pragma unroll
    for (int w = 0; w < 8; w++) {
        unsigned word = __ballot_sync(0xffffffffu, (m >> w) & 1u);
        if (lane == w) mine = word;
    }
    if (lane < 8) plane[b * 8 + lane] = mine;
}

// ---------------------------------------------------------------- exclusion masks (a4)
struct ExclArgs {
    int natoms;
    const int *excl_off, *excl_idx, *slot_of_atom, *ent_count, *ent_jbegin;
    int2* jl;
    const uint8_t* imask;
    unsigned long long* masks;
};

// One thread per atom; each unordered excluded pair is handled once (from its lower index), in
// both orientations and under every shift the cluster pair is listed with (S:8.3.2 pairmask).
// MODE 0 marks the joint entries that need a mask, MODE 1 clears the pair bits.
// Internal bit index is b*8+a (transposed w.r.t. the ABI's a*8+b) so that the lane owning
// j-atom b reads its 8 i-atom bits as one byte.
template <int MODE>
__global__ void k_excl(ExclArgs A)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= A.natoms) return;
    for (int e = A.excl_off[i]; e < A.excl_off[i + 1]; e++) {
        int j = A.excl_idx[e];
        if (j <= i) continue;
        int sl[2] = {A.slot_of_atom[i], A.slot_of_atom[j]};
#pragma unroll
        for (int o = 0; o < 2; o++) {
            int p = sl[o], q = sl[1 - o];
            int cp = p >> 3, cq = q >> 3, a = p & 7, b = q & 7;
            int scp = cp >> 3, w = cp & 7;
            for (int h = 0; h < NB_NHALF; h++) {
                int ent = scp * NB_NHALF + h;
                int cnt = A.ent_count[ent];
                if (cnt == 0) continue;
                int lo = A.ent_jbegin[ent], hi = lo + cnt;
                while (lo < hi) {
                    int mid = (lo + hi) >> 1;
                    if (A.jl[mid].x < cq) lo = mid + 1; else hi = mid;
                }
                if (lo < A.ent_jbegin[ent] + cnt && A.jl[lo].x == cq && ((A.imask[lo] >> w) & 1)) {
                    if (MODE == 0) A.jl[lo].y = 1;
                    else atomicAnd(&A.masks[((size_t)A.jl[lo].y * 8 + w) * 2], ~(1ull << (b * 8 + a)));
                }
            }
        }
    }
}

__global__ void k_excl_flags(const int2* __restrict__ jl, int* __restrict__ flag, long long n)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) flag[i] = jl[i].y != 0 ? 1 : 0;
}

// Assigns mask refs (1-based; 0 = "no mask") and initialises the masks: all pairs interact,
// except on the diagonal cluster pair (cj == ci at zero shift) where only b > a is counted.
__global__ void k_excl_assign(int2* __restrict__ jl, const int* __restrict__ prefix, const int* __restrict__ batch_ent,
                              unsigned long long* __restrict__ masks, long long n)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) {
        for (int w = 0; w < 16; w++) masks[w] = ~0ull;
    }
    if (i >= n) return;
    int2 e = jl[i];
    if (e.y == 0) return;
    int ref = prefix[i] + 1;
    jl[i].y = ref;
    int ent = batch_ent[i >> 5];
    int sci = ent / NB_NHALF, h = ent % NB_NHALF;
    unsigned long long upper = 0;   // bit b*8+a set iff b > a
    for (int b = 0; b < 8; b++)
        for (int a = 0; a < b; a++) upper |= 1ull << (b * 8 + a);
    for (int w = 0; w < 8; w++) {
        bool diag = h == 0 && e.x == sci * 8 + w;
        masks[((size_t)ref * 8 + w) * 2] = diag ? upper : ~0ull;       // interact
        masks[((size_t)ref * 8 + w) * 2 + 1] = diag ? upper : ~0ull;   // counted at all
    }
}

// One warp per batch of 32 joint entries: word (batch, w) of plane_excl has bit e set iff entry e
// carries a mask whose row for i-cluster w is not all-ones (a force-field exclusion, a self pair
// or the lower triangle of a diagonal cluster pair).  The force kernel routes exactly those
// (entry, i-cluster) pairs through its masked instantiation.
__global__ void k_excl_planes(const int2* __restrict__ jl, const unsigned long long* __restrict__ masks,
                              uint32_t* __restrict__ plane_excl, long long nbatch)
{
    long long b = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (b >= nbatch) return;
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

// ---------------------------------------------------------------- compact inner list (nb_internal.h)
// Segment capacities per (work unit, i-cluster): every outer cluster pair can survive a prune.
__global__ void k_ilist_caps(const int4* __restrict__ units, int nunits, const uint32_t* __restrict__ plane_outer,
                             const uint32_t* __restrict__ plane_excl, int* __restrict__ capu, int* __restrict__ capm)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nunits * 8) return;
    const int4 u = units[i >> 3];
    const int w = i & 7;
    int nu = 0, nm = 0;
    for (int b = u.y; b < u.z; b++) {
        const unsigned bits = plane_outer[(size_t)b * 8 + w], eb = plane_excl[(size_t)b * 8 + w] & bits;
        nu += __popc(bits & ~eb);
        nm += __popc(eb);
    }
    capu[i] = (2 * nu + 7) & ~7;   // half-cluster entries, multiple of 8
    capm[i] = nm;
}

// After a search, one block per work unit (launch order): inner := outer.
__global__ void __launch_bounds__(256) k_ilist_build(const int4* __restrict__ units, const uint32_t* __restrict__ plane,
                                                     const uint32_t* __restrict__ plane_excl, const int2* __restrict__ jl,
                                                     const int* __restrict__ il_off, const int* __restrict__ ilm_off,
                                                     const int* __restrict__ seg_pos, int4* __restrict__ seg,
                                                     int2* __restrict__ seg_ci, int32_t* __restrict__ il,
                                                     int2* __restrict__ ilm, int2* __restrict__ ol, int2* __restrict__ ol_cnt,
                                                     int cj_dummy)
{
    const int4 u = units[blockIdx.x];   // units in launch order
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, s0 = blockIdx.x * 8 + warp;
    const int o = il_off[s0], om = ilm_off[s0];
    const int s = seg_pos[s0];
    if (lane == 0) {
        seg[s].x = o;
        seg[s].y = om;
        seg_ci[s] = make_int2(u.w * 8 + warp, nb_half_shift_id(u.x - u.w * NB_NHALF));
    }
    {   // compact outer list of this i-cluster, what the prune kernel streams: the cluster pairs
        // without a mask first, then (from a multiple of 4 on) those with a mask
        int2* ols = ol + o + om;
        const unsigned lt = (1u << lane) - 1u;
        int nuo = 0, nmo = 0;
        for (int b = u.y; b < u.z; b++) {
            const unsigned bits = plane[(size_t)b * 8 + warp], eb = plane_excl[(size_t)b * 8 + warp] & bits;
            nuo += __popc(bits & ~eb);
        }
        const int mbase = (nuo + 3) & ~3;
        nuo = 0;
        for (int b = u.y; b < u.z; b++) {
            const unsigned bits = plane[(size_t)b * 8 + warp], eb = plane_excl[(size_t)b * 8 + warp] & bits, nb = bits & ~eb;
            if ((bits >> lane) & 1u) {
                const int2 e = make_int2(jl[(size_t)b * 32 + lane].x, (b - u.y) * 32 + lane);
                if ((nb >> lane) & 1u) ols[nuo + __popc(nb & lt)] = e;
                else ols[mbase + nmo + __popc(eb & lt)] = e;
            }
            nuo += __popc(nb);
            nmo += __popc(eb);
        }
        if (lane == 0) ol_cnt[s0] = make_int2(nuo, nmo);
    }
    nb_ilist_write([&](int b) { return plane[(size_t)(u.y + b) * 8 + warp]; }, u.y, u.z, warp, lane, cj_dummy, plane_excl, jl,
                   il + o, ilm + om, reinterpret_cast<int2*>(&seg[s]) + 1);
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

__device__ __forceinline__ unsigned entry_bits(const uint32_t* plane, long long e)
{
    unsigned bits = 0;
    const uint32_t* p = plane + (e >> 5) * 8;
#pragma unroll
    for (int w = 0; w < 8; w++) bits |= ((p[w] >> (e & 31)) & 1u) << w;
    return bits;
}

__global__ void k_dump_count(const uint32_t* __restrict__ plane, int* __restrict__ cnt, long long n)
{
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < n) cnt[e] = __popc(entry_bits(plane, e));
}

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
    int sci = ent / NB_NHALF, h = ent % NB_NHALF;
    int u = A.batch_unit[e >> 5];
    int part = (int)(((long long)u * A.nparts) / A.nunits);
    while (part + 1 < A.nparts && ((long long)(part + 1) * A.nunits) / A.nparts <= u) part++;
    while (part > 0 && ((long long)part * A.nunits) / A.nparts > u) part--;
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

}  // namespace

int nbi_exclusive_scan(nb_ctx* c, const int32_t* in, int32_t* out, int64_t n, int32_t* total_dev)
{
    if (n <= 0) {
        if (total_dev) NB_CUDA(c, cudaMemsetAsync(total_dev, 0, sizeof(int), c->stream));
        return NB_OK;
    }
    int nblk = (int)((n + 1023) / 1024);
    NB_CUDA(c, c->scan_blk.ensure(nblk + 1, c->stream));
    k_scan1<<<nblk, 1024, 0, c->stream>>>(in, out, c->scan_blk.p, n);
    NB_LAUNCH_CHECK(c);
    k_scan2<<<1, 1024, 0, c->stream>>>(c->scan_blk.p, nblk, total_dev);
    NB_LAUNCH_CHECK(c);
    k_scan3<<<nblk, 1024, 0, c->stream>>>(out, c->scan_blk.p, n);
    NB_LAUNCH_CHECK(c);
    return NB_OK;
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

int nbi_list_count(nb_ctx* c, int which, int64_t* n)
{
    return count_bits(c, which == 0 ? c->plane_outer.p : c->plane_inner.p, n);
}

int nbi_search(nb_ctx* c, float rlist)
{
    cudaStream_t st = c->stream;
    int rc = nbi_grid(c);
    if (rc != NB_OK) return rc;
    const int nsc = c->nsc;
    NbStageTimer* tm = new NbStageTimer(c, NB_T_SEARCH);
    struct TmGuard { NbStageTimer*& t; ~TmGuard() { delete t; } } tm_guard{tm};
    c->nent = nsc * NB_NHALF;
    NB_CUDA(c, c->ent_count.ensure(c->nent + 1, st));
    NB_CUDA(c, c->ent_jbegin.ensure(c->nent + 1, st));

    SearchArgs A;
    A.nsc = nsc; A.ncx = c->ncx; A.ncy = c->ncy; A.inv_cx = c->inv_cx; A.inv_cy = c->inv_cy;
    for (int k = 0; k < 3; k++) A.box[k] = c->box[k];
    A.rl2 = rlist * rlist;
    A.rm = rlist * (1.0f + 1e-5f) + 1e-5f;
    A.rm2 = A.rm * A.rm;
    A.col_sc_off = c->col_sc_off.p;
    A.sbb_lo = c->sbb_lo.p; A.sbb_hi = c->sbb_hi.p; A.bb_lo = c->bb_lo.p; A.bb_hi = c->bb_hi.p;
    A.ent_count = c->ent_count.p; A.ent_jbegin = nullptr; A.jl = nullptr; A.imask = nullptr;
    k_search<false><<<(nsc + 3) / 4, 128, 0, st>>>(A);
    NB_LAUNCH_CHECK(c);

    // Host side of (a5): element offsets (32-aligned), split into bounded work units, order.
    c->h_ent_count.resize(c->nent);
    c->h_ent_jbegin.resize(c->nent + 1);
    NB_CUDA(c, cudaMemcpyAsync(c->h_ent_count.data(), c->ent_count.p, sizeof(int) * c->nent, cudaMemcpyDeviceToHost, st));
    NB_CUDA(c, cudaStreamSynchronize(st));
    int64_t off = 0, nent_nonempty = 0;
    for (int e = 0; e < c->nent; e++) {
        c->h_ent_jbegin[e] = (int32_t)off;
        int cnt = c->h_ent_count[e];
        if (cnt) nent_nonempty++;
        off += ((int64_t)cnt + NB_BATCH - 1) / NB_BATCH * NB_BATCH;
        if (off > 0x7fffff00LL) return nb_fail(c, NB_ERR_OVERFLOW, "pair list exceeds 2^31 joint entries");
    }
    c->h_ent_jbegin[c->nent] = (int32_t)off;
    c->njslots = off;
    c->nbatch = off / NB_BATCH;

    // L199-L201: "heuristically split lists to increase the available parallelism": a work unit is
    // at most `ub` batches of one element; `ub` is chosen so that there are about 16 units per SM.
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, c->prm.device);
    int per_sm = 6;
    if (const char* e = getenv("NB_UNITS_PER_SM")) per_sm = std::max(1, atoi(e));   // tuning knob
    int64_t target = (int64_t)per_sm * nsm;
    int ub = (int)std::min<int64_t>(NB_MAX_UNIT_BATCHES, std::max<int64_t>(1, c->nbatch / target));
    c->h_units.clear();
    std::vector<int32_t> h_batch_ent(c->nbatch), h_batch_unit(c->nbatch);
    for (int e = 0; e < c->nent; e++) {
        int cnt = c->h_ent_count[e];
        if (!cnt) continue;
        int b0 = c->h_ent_jbegin[e] / NB_BATCH, nb = (cnt + NB_BATCH - 1) / NB_BATCH;
        const int nsplit = (nb + ub - 1) / ub;   // equal-sized chunks of at most ub batches
        for (int k = 0; k < nsplit; k++) {
            const int b = (int)((int64_t)nb * k / nsplit), bend = (int)((int64_t)nb * (k + 1) / nsplit);
            for (int bb = b; bb < bend; bb++) {
                h_batch_ent[b0 + bb] = e;
                h_batch_unit[b0 + bb] = (int)c->h_units.size();
            }
            c->h_units.push_back(make_int4(e, b0 + b, b0 + bend, e / NB_NHALF));
        }
    }
    c->nunits = (int)c->h_units.size();
    // L199: "reshaped by sorting to avoid long lists being scheduled late": longest units first
    // (stable, so the order is deterministic).
    std::vector<int4> sorted(c->h_units);
    std::stable_sort(sorted.begin(), sorted.end(),
                     [](const int4& a, const int4& b) { return (a.z - a.y) > (b.z - b.y); });
    std::vector<int32_t> order(c->nunits), pos(c->nunits);
    for (int i = 0; i < c->nunits; i++) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
        return (c->h_units[a].z - c->h_units[a].y) > (c->h_units[b].z - c->h_units[b].y);
    });
    for (int i = 0; i < c->nunits; i++) pos[order[i]] = i;
    c->h_unit_order = order;

    NB_CUDA(c, c->jl.ensure(std::max<int64_t>(c->njslots, 1), st));
    NB_CUDA(c, c->imask_outer.ensure(std::max<int64_t>(c->njslots, 1), st));
    NB_CUDA(c, c->plane_outer.ensure(std::max<int64_t>(c->nbatch * 8, 1), st));
    NB_CUDA(c, c->plane_inner.ensure(std::max<int64_t>(c->nbatch * 8, 1), st));
    NB_CUDA(c, c->plane_excl.ensure(std::max<int64_t>(c->nbatch * 8, 1), st));
    NB_CUDA(c, c->batch_ent.ensure(std::max<int64_t>(c->nbatch, 1) * 2, st));
    NB_CUDA(c, c->units_canon.ensure(std::max(c->nunits, 1), st));
    NB_CUDA(c, c->units_sorted.ensure(std::max(c->nunits, 1), st));
    NB_CUDA(c, c->unit_order.ensure(std::max(c->nunits, 1), st));
    NB_CUDA(c, c->unit_pos.ensure(std::max(c->nunits, 1), st));
    NB_CUDA(c, c->scan_tmp.ensure(std::max<int64_t>(c->njslots, 1) * 2 + 8, st));
    NB_CUDA(c, cudaMemcpyAsync(c->ent_jbegin.p, c->h_ent_jbegin.data(), sizeof(int) * (c->nent + 1), cudaMemcpyHostToDevice, st));
    int* d_batch_unit = c->batch_ent.p + std::max<int64_t>(c->nbatch, 1);
    if (c->nbatch) {
        NB_CUDA(c, cudaMemcpyAsync(c->batch_ent.p, h_batch_ent.data(), sizeof(int) * c->nbatch, cudaMemcpyHostToDevice, st));
        NB_CUDA(c, cudaMemcpyAsync(d_batch_unit, h_batch_unit.data(), sizeof(int) * c->nbatch, cudaMemcpyHostToDevice, st));
        NB_CUDA(c, cudaMemcpyAsync(c->units_canon.p, c->h_units.data(), sizeof(int4) * c->nunits, cudaMemcpyHostToDevice, st));
        NB_CUDA(c, cudaMemcpyAsync(c->units_sorted.p, sorted.data(), sizeof(int4) * c->nunits, cudaMemcpyHostToDevice, st));
        NB_CUDA(c, cudaMemcpyAsync(c->unit_order.p, order.data(), sizeof(int) * c->nunits, cudaMemcpyHostToDevice, st));
        NB_CUDA(c, cudaMemcpyAsync(c->unit_pos.p, pos.data(), sizeof(int) * c->nunits, cudaMemcpyHostToDevice, st));
        NB_CUDA(c, cudaMemsetAsync(c->imask_outer.p, 0, c->njslots, st));
        k_init_jl<<<(unsigned)((c->njslots + 255) / 256), 256, 0, st>>>(c->jl.p, c->njslots);
        NB_LAUNCH_CHECK(c);
    }
    A.ent_jbegin = c->ent_jbegin.p; A.jl = c->jl.p; A.imask = c->imask_outer.p;
    k_search<true><<<(nsc + 3) / 4, 128, 0, st>>>(A);
    NB_LAUNCH_CHECK(c);
    if (c->nbatch) {
        k_planes<<<(unsigned)((c->nbatch * 32 + 255) / 256), 256, 0, st>>>(c->imask_outer.p, c->plane_outer.p, c->nbatch);
        NB_LAUNCH_CHECK(c);
        NB_CUDA(c, cudaMemcpyAsync(c->plane_inner.p, c->plane_outer.p, sizeof(uint32_t) * c->nbatch * 8, cudaMemcpyDeviceToDevice, st));
    }

    // (a4) exclusion masks
    delete tm;
    tm = new NbStageTimer(c, NB_T_MASKS);
    ExclArgs E;
    E.natoms = c->natoms; E.excl_off = c->excl_off.p; E.excl_idx = c->excl_idx.p; E.slot_of_atom = c->slot_of_atom.p;
    E.ent_count = c->ent_count.p; E.ent_jbegin = c->ent_jbegin.p; E.jl = c->jl.p; E.imask = c->imask_outer.p;
    E.masks = nullptr;
    if (c->nexcl && c->nbatch) {
        k_excl<0><<<(c->natoms + 127) / 128, 128, 0, st>>>(E);
        NB_LAUNCH_CHECK(c);
    }
    int* flag = c->scan_tmp.p;
    int* prefix = c->scan_tmp.p + std::max<int64_t>(c->njslots, 1);
    int* total_dev = c->scan_tmp.p + 2 * std::max<int64_t>(c->njslots, 1);
    int nmask = 0;
    if (c->nbatch) {
        k_excl_flags<<<(unsigned)((c->njslots + 255) / 256), 256, 0, st>>>(c->jl.p, flag, c->njslots);
        NB_LAUNCH_CHECK(c);
        rc = nbi_exclusive_scan(c, flag, prefix, c->njslots, total_dev);
        if (rc != NB_OK) return rc;
        NB_CUDA(c, cudaMemcpyAsync(&nmask, total_dev, sizeof(int), cudaMemcpyDeviceToHost, st));
        NB_CUDA(c, cudaStreamSynchronize(st));
    }
    c->nmask = nmask;
    NB_CUDA(c, c->excl_masks.ensure((size_t)(nmask + 1) * 16, st));
    if (c->nbatch) {
        k_excl_assign<<<(unsigned)((c->njslots + 255) / 256), 256, 0, st>>>(c->jl.p, prefix, c->batch_ent.p, c->excl_masks.p, c->njslots);
        NB_LAUNCH_CHECK(c);
        if (c->nexcl) {
            E.masks = c->excl_masks.p;
            k_excl<1><<<(c->natoms + 127) / 128, 128, 0, st>>>(E);
            NB_LAUNCH_CHECK(c);
        }
        k_excl_planes<<<(unsigned)((c->nbatch * 32 + 255) / 256), 256, 0, st>>>(c->jl.p, c->excl_masks.p, c->plane_excl.p, c->nbatch);
        NB_LAUNCH_CHECK(c);
        // compact inner list: segment offsets from the outer counts, then inner := outer
        const int nseg = c->nunits * 8;
        NB_CUDA(c, c->il_off.ensure(nseg, st));
        NB_CUDA(c, c->ilm_off.ensure(nseg, st));
        NB_CUDA(c, c->seg.ensure(nseg, st));
        int* capu = c->scan_tmp.p;
        int* capm = c->scan_tmp.p + nseg;
        k_ilist_caps<<<(nseg + 255) / 256, 256, 0, st>>>(c->units_sorted.p, c->nunits, c->plane_outer.p, c->plane_excl.p, capu, capm);
        NB_LAUNCH_CHECK(c);
        rc = nbi_exclusive_scan(c, capu, c->il_off.p, nseg, total_dev);
        if (rc != NB_OK) return rc;
        rc = nbi_exclusive_scan(c, capm, c->ilm_off.p, nseg, total_dev + 1);
        if (rc != NB_OK) return rc;
        int tot[2] = {0, 0};
        NB_CUDA(c, cudaMemcpyAsync(tot, total_dev, sizeof(tot), cudaMemcpyDeviceToHost, st));
        c->h_caps.resize((size_t)2 * nseg);
        NB_CUDA(c, cudaMemcpyAsync(c->h_caps.data(), capu, sizeof(int) * 2 * nseg, cudaMemcpyDeviceToHost, st));
        NB_CUDA(c, cudaStreamSynchronize(st));
        {
            // L199: longest lists first, now per i-cluster list: counting sort of the segments by
            // outer length (descending, stable); empty segments are not launched.
            const int* cu = c->h_caps.data();
            const int* cm = cu + nseg;
            int maxlen = 0;
            for (int i = 0; i < nseg; i++) maxlen = std::max(maxlen, cu[i] + 2 * cm[i]);
            std::vector<int32_t> start(maxlen + 2, 0);
            std::vector<int32_t>& pos = c->h_seg_pos;   // member: source of an async upload
            pos.resize(nseg);
            for (int i = 0; i < nseg; i++) start[maxlen - (cu[i] + 2 * cm[i]) + 1]++;
            for (int l = 0; l <= maxlen; l++) start[l + 1] += start[l];
            c->nseg_launch = start[maxlen];   // everything before the length-0 bucket
            for (int i = 0; i < nseg; i++) pos[i] = start[maxlen - (cu[i] + 2 * cm[i])]++;
            c->h_seg_sorted.resize(nseg);   // sorted position -> (unit launch position*8 + i-cluster)
            for (int i = 0; i < nseg; i++) c->h_seg_sorted[pos[i]] = i;
            NB_CUDA(c, c->seg_pos.ensure(nseg, st));
            NB_CUDA(c, c->seg_ci.ensure(nseg, st));
            NB_CUDA(c, cudaMemcpyAsync(c->seg_pos.p, pos.data(), sizeof(int) * nseg, cudaMemcpyHostToDevice, st));
        }
        c->il_total = (size_t)tot[0];
        c->ilm_total = (size_t)tot[1];
        NB_CUDA(c, c->il.ensure((size_t)tot[0] + 4, st));
        NB_CUDA(c, c->ilm.ensure((size_t)tot[1] + 4, st));
        NB_CUDA(c, c->ol.ensure((size_t)tot[0] + (size_t)tot[1] + 4, st));
        NB_CUDA(c, c->ol_cnt.ensure(nseg, st));
        k_ilist_build<<<c->nunits, 256, 0, st>>>(c->units_sorted.p, c->plane_inner.p, c->plane_excl.p, c->jl.p, c->il_off.p,
                                                 c->ilm_off.p, c->seg_pos.p, c->seg.p, c->seg_ci.p, c->il.p, c->ilm.p, c->ol.p, c->ol_cnt.p, c->nclusters);
        NB_LAUNCH_CHECK(c);
    } else {
        std::vector<unsigned long long> ones(16, ~0ull);
        NB_CUDA(c, cudaMemcpyAsync(c->excl_masks.p, ones.data(), 16 * sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
        NB_CUDA(c, cudaStreamSynchronize(st));
    }

    // statistics
    NB_CUDA(c, c->counters.ensure(8, st));
    NB_CUDA(c, cudaMemsetAsync(c->counters.p, 0, 8 * sizeof(long long), st));
    if (c->nbatch) {
        k_count_bits<<<(unsigned)((c->nbatch * 8 + 255) / 256), 256, 0, st>>>(c->plane_outer.p, c->nbatch * 8, c->counters.p);
        NB_LAUNCH_CHECK(c);
        k_count_joint<<<(unsigned)((c->njslots + 255) / 256), 256, 0, st>>>(c->imask_outer.p, c->jl.p, c->njslots, c->counters.p + 1);
        NB_LAUNCH_CHECK(c);
    }
    long long cnt[3] = {0, 0, 0};
    NB_CUDA(c, cudaMemcpyAsync(cnt, c->counters.p, sizeof(cnt), cudaMemcpyDeviceToHost, st));
    NB_CUDA(c, cudaStreamSynchronize(st));
    c->st.n_sci_entries = nent_nonempty;
    c->st.n_pairs_outer = cnt[0];
    c->st.n_pairs_inner = cnt[0];
    c->st.n_joint_outer = cnt[1];
    c->st.n_excl_masks = cnt[2];
    c->st.n_work_units = c->nunits;
    c->rlist_outer = rlist;
    c->last_nparts = 1;
    c->have_list = true;
    c->st.search_count++;
    return NB_OK;
}

int nbi_list_dump(nb_ctx* c, int which, int32_t* ci, int32_t* cj, int32_t* shift, uint64_t* pairmask, int32_t* part)
{
    if (!c->nbatch) return NB_OK;
    cudaStream_t st = c->stream;
    const uint32_t* plane = which == 0 ? c->plane_outer.p : c->plane_inner.p;
    int* cnt = c->scan_tmp.p;
    int* off = c->scan_tmp.p + c->njslots;
    k_dump_count<<<(unsigned)((c->njslots + 255) / 256), 256, 0, st>>>(plane, cnt, c->njslots);
    NB_LAUNCH_CHECK(c);
    int rc = nbi_exclusive_scan(c, cnt, off, c->njslots, nullptr);
    if (rc != NB_OK) return rc;
    DumpArgs D;
    D.plane = plane; D.offset = off; D.jl = c->jl.p; D.batch_ent = c->batch_ent.p;
    D.batch_unit = c->batch_ent.p + std::max<int64_t>(c->nbatch, 1);
    D.atom_of_slot = c->atom_of_slot.p; D.masks = c->excl_masks.p; D.n = c->njslots;
    D.nunits = std::max(c->nunits, 1); D.nparts = std::max(c->last_nparts, 1);
    D.ci = ci; D.cj = cj; D.shift = shift; D.part = part; D.pairmask = pairmask;
    k_dump_fill<<<(unsigned)((c->njslots + 255) / 256), 256, 0, st>>>(D);
    NB_LAUNCH_CHECK(c);
    NB_CUDA(c, cudaStreamSynchronize(st));
    return NB_OK;
}
