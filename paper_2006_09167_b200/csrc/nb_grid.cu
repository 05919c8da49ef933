// nb_grid.cu -- (a1) coordinate refresh and (a2) gridding + cluster sort.
//
// "The clusters and pair list are obtained during search using a regular grid in
// x and y dimensions but binning the resulting z columns into cells with fixed number of
// particles"; L131: super-clusters come from "a 2x2x2 cell grouping on the search grid".
// The paper does this on the CPU; here it runs on the GPU (BASELINE.json north_star: one GPU,
// no CPU fallback).  Readings A10/A11: column side ~ (64/rho)^(1/3); per column a
// z-sort, 64-atom slabs, each split by y (2x32), x (2x16), z (2x8), ties by atom index; a
// partly filled last slab fills its clusters in that order, real atoms first.
#include "nb_internal.h"

#include <math.h>

namespace {

__device__ __forceinline__ uint32_t float_orderable(float v)
{
    uint32_t u = __float_as_uint(v);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// One thread per atom: wrap into the box (image fixed until the next search), column index,
// rank inside the column (arrival order; the later sort makes the layout deterministic).
// The column counters are few (a hundred for 100k atoms) and consecutive atoms mostly share a column,
// so the lanes of a warp that hit the same column send ONE atomic (match_any + popc ranks).
__global__ void k_bin(int n, const float* __restrict__ x, const float* __restrict__ q, const int* __restrict__ type,
                      int ntypes, float3 box, int ncx, int ncy, float inv_cx, float inv_cy, int nlocal, char4* __restrict__ image,
                      float4* __restrict__ xw_atom, int* __restrict__ atom_col, int* __restrict__ atom_rank,
                      int* __restrict__ col_count, NbTotals* __restrict__ tot)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    int col = -1;
    if (i < n) {
        float L[3] = {box.x, box.y, box.z};
        float w[3];
        int img[3];
#pragma unroll
        for (int k = 0; k < 3; k++) {
            float v = x[3 * i + k];
            float kf = floorf(v / L[k]);
            float t = __fmaf_rn(-kf, L[k], v);
            if (t < 0.f) { kf -= 1.f; t = __fmaf_rn(-kf, L[k], v); }
            else if (t >= L[k]) { kf += 1.f; t = __fmaf_rn(-kf, L[k], v); }
            kf = fminf(fmaxf(kf, -127.f), 127.f);
            w[k] = __fmaf_rn(-kf, L[k], v);
            img[k] = (int)kf;
        }
        int cx = min(ncx - 1, max(0, (int)floorf(w[0] * inv_cx)));
        int cy = min(ncy - 1, max(0, (int)floorf(w[1] * inv_cy)));
        col = cx * ncy + cy + (i >= nlocal ? ncx * ncy : 0);   // non-local atoms: the second column set (nb_set_local)
        image[i] = make_char4((signed char)img[0], (signed char)img[1], (signed char)img[2], 0);
        xw_atom[i] = make_float4(w[0], w[1], w[2], q[i]);
        atom_col[i] = col;
        const int t = type[i];
        if (t < 0 || t >= ntypes) tot->bad_type = 1;   // reported as NB_ERR_ARG at the end of the search
    }
    const unsigned peers = __match_any_sync(0xffffffffu, col);
    if (col >= 0) {
        const int leader = __ffs(peers) - 1;
        int base = 0;
        if (lane == leader) base = atomicAdd(&col_count[col], __popc(peers));
        base = __shfl_sync(peers, base, leader);
        atom_rank[i] = base + __popc(peers & ((1u << lane) - 1u));
    }
}

// Single block: exclusive scans over columns of the atom count and of the super-cluster count.
__global__ void k_col_scan(int ncol, int ncol_local, const int* __restrict__ col_count, int* __restrict__ col_atom_off,
                           int* __restrict__ col_sc_off, NbTotals* __restrict__ totals)
{
    __shared__ int s_a[1024], s_s[1024];
    __shared__ int carry_a, carry_s, maxc;
    int t = threadIdx.x;
    if (t == 0) { carry_a = 0; carry_s = 0; maxc = 0; }
    __syncthreads();
    for (int base = 0; base < ncol; base += 1024) {
        int c = base + t;
        int cnt = c < ncol ? col_count[c] : 0;
        int nsc = (cnt + NB_SC_ATOMS - 1) / NB_SC_ATOMS;
        s_a[t] = cnt;
        s_s[t] = nsc;
        atomicMax(&maxc, cnt);
        __syncthreads();
        for (int d = 1; d < 1024; d <<= 1) {
            int va = t >= d ? s_a[t - d] : 0, vs = t >= d ? s_s[t - d] : 0;
            __syncthreads();
            s_a[t] += va;
            s_s[t] += vs;
            __syncthreads();
        }
        if (c < ncol) {
            col_atom_off[c] = carry_a + s_a[t] - cnt;
            col_sc_off[c] = carry_s + s_s[t] - nsc;
            if (c == ncol_local) totals->nsc_local = carry_s + s_s[t] - nsc;   // first super-cluster of the non-local columns
        }
        __syncthreads();
        if (t == 1023) { carry_a += s_a[t]; carry_s += s_s[t]; }
        __syncthreads();
    }
    if (t == 0) {
        col_atom_off[ncol] = carry_a;
        col_sc_off[ncol] = carry_s;
        totals->nsc = carry_s;
        if (ncol_local >= ncol) totals->nsc_local = carry_s;
        totals->max_col = maxc;
    }
}

__global__ void k_col_scatter(int n, const int* __restrict__ atom_col, const int* __restrict__ atom_rank,
                              const int* __restrict__ col_atom_off, int* __restrict__ col_atoms)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    col_atoms[col_atom_off[atom_col[i]] + atom_rank[i]] = i;
}

struct SlabScratch {
    float key[NB_SC_ATOMS];
    int atom[NB_SC_ATOMS];
    int atom2[NB_SC_ATOMS];
};

// Stable rank sort of the 64 entries of a slab inside segments of `seg` entries, by
// (coordinate `comp`, atom index); invalid entries (atom == INT_MAX) sort last.
__device__ __forceinline__ void slab_segment_sort(SlabScratch& s, const float4* __restrict__ xw_atom, int comp,
                                                  int seg, int lane)
{
#pragma unroll
    for (int h = 0; h < 2; h++) {
        int e = lane + 32 * h;
        int a = s.atom[e];
        float4 v = a != INT_MAX ? xw_atom[a] : make_float4(INFINITY, INFINITY, INFINITY, 0.f);
        s.key[e] = comp == 0 ? v.x : (comp == 1 ? v.y : v.z);
    }
    __syncwarp();
#pragma unroll
    for (int h = 0; h < 2; h++) {
        int e = lane + 32 * h;
        int s0 = (e / seg) * seg;
        float k = s.key[e];
        int a = s.atom[e];
        int rank = 0;
        for (int o = s0; o < s0 + seg; o++) {
            float ko = s.key[o];
            int ao = s.atom[o];
            rank += (ko < k || (ko == k && (ao < a || (ao == a && o < e)))) ? 1 : 0;   // padding entries tie: keep order
        }
        s.atom2[s0 + rank] = a;
    }
    __syncwarp();
#pragma unroll
    for (int h = 0; h < 2; h++) s.atom[lane + 32 * h] = s.atom2[lane + 32 * h];
    __syncwarp();
}

// One block per grid column: bitonic z-sort of the column in shared memory, then one warp per
// 64-atom slab does the 2x2x2 sub-sorts and writes the cluster-ordered arrays and bounding boxes.
#define NB_LAYOUT_WARPS 16   // warps per column block: one per 64-atom slab in flight (a column of config 2 holds 13 slabs)
__global__ void __launch_bounds__(32 * NB_LAYOUT_WARPS)
k_col_layout(int ncy, int ncol_local, const int* __restrict__ col_atom_off, const int* __restrict__ col_sc_off,
             const int* __restrict__ col_atoms, const float4* __restrict__ xw_atom,
             const int* __restrict__ type, int pad_type, int np2_max, float4* __restrict__ xq,
             int* __restrict__ type_slot, int* __restrict__ atom_of_slot, int* __restrict__ slot_of_atom,
             float4* __restrict__ bb_lo, float4* __restrict__ bb_hi, float4* __restrict__ sbb_lo,
             float4* __restrict__ sbb_hi, float3 pad_base, float3 pad_step, NbTotals* __restrict__ tot)
{
    extern __shared__ unsigned long long s_keys[];
    __shared__ SlabScratch s_slab[NB_LAYOUT_WARPS];
    int col = blockIdx.x;
    int a0 = col_atom_off[col], n = col_atom_off[col + 1] - a0;
    if (n == 0) return;
    if (n > np2_max) {   // the sort buffer was sized from the previous search: say so, the host repeats the search
        if (threadIdx.x == 0) atomicOr(&tot->overflow, NB_OVF_COL);
        return;
    }
    int np2 = 1;
    while (np2 < n) np2 <<= 1;
    for (int i = threadIdx.x; i < np2; i += blockDim.x) {
        unsigned long long k = ~0ull;
        if (i < n) {
            int a = col_atoms[a0 + i];
            k = ((unsigned long long)float_orderable(xw_atom[a].z) << 32) | (unsigned)a;
        }
        s_keys[i] = k;
    }
    __syncthreads();
    for (int k = 2; k <= np2; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int i = threadIdx.x; i < np2; i += blockDim.x) {
                int p = i ^ j;
                if (p > i) {
                    unsigned long long u = s_keys[i], v = s_keys[p];
                    bool up = (i & k) == 0;
                    if ((u > v) == up) { s_keys[i] = v; s_keys[p] = u; }
                }
            }
            __syncthreads();
        }
    }
    int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int nslab = (n + NB_SC_ATOMS - 1) / NB_SC_ATOMS;
    int sc0 = col_sc_off[col];
    SlabScratch& s = s_slab[warp];
    for (int slab = warp; slab < nslab; slab += NB_LAYOUT_WARPS) {
#pragma unroll
        for (int h = 0; h < 2; h++) {
            int e = lane + 32 * h, idx = slab * NB_SC_ATOMS + e;
            s.atom[e] = idx < n ? (int)(unsigned)(s_keys[idx] & 0xffffffffull) : INT_MAX;
        }
        __syncwarp();
        slab_segment_sort(s, xw_atom, 1, 64, lane);   // y: 2 x 32
        slab_segment_sort(s, xw_atom, 0, 32, lane);   // x: 2 x 16
        slab_segment_sort(s, xw_atom, 2, 16, lane);   // z: 2 x 8 -> clusters of 8
        int sc = sc0 + slab;
        float slo[3] = {1e30f, 1e30f, 1e30f}, shi[3] = {-1e30f, -1e30f, -1e30f};
#pragma unroll
        for (int h = 0; h < 2; h++) {
            int e = lane + 32 * h;
            int slot = sc * NB_SC_ATOMS + e;
            int a = s.atom[e];
            bool real = a != INT_MAX;
            float4 v;
            if (real) {
                v = xw_atom[a];
                slot_of_atom[a] = slot;
            } else {
                // padding (reading A11): zero charge, zero-LJ type, outside every cut-off of every
                // real atom under every shift (x < -(2 Lx + 8)), distinct per (slot, column mod 64)
                // with a spacing d_k chosen so that L_k / d_k is a half-integer: two padding atoms
                // never coincide under any shift, and all distances stay small enough (< ~1e3 nm)
                // for the force kernel's arithmetic to remain finite without a clamp.
                // (the padding of a non-local column, which lies on top of its local twin, sits 128 lattice steps further out)
                const int cls = col >= ncol_local ? 1 : 0, colm = col - cls * ncol_local;
                int cx = colm / ncy, cy = colm % ncy;
                v = make_float4(pad_base.x - pad_step.x * (float)(e + 128 * cls), pad_base.y - pad_step.y * (float)(cy & 63),
                                pad_base.z - pad_step.z * (float)(cx & 63), 0.f);
            }
            xq[slot] = v;
            type_slot[slot] = real ? type[a] : pad_type;
            atom_of_slot[slot] = real ? a : -1;
            float lo[3] = {real ? v.x : 1e30f, real ? v.y : 1e30f, real ? v.z : 1e30f};
            float hi[3] = {real ? v.x : -1e30f, real ? v.y : -1e30f, real ? v.z : -1e30f};
            int cnt = real ? 1 : 0;
#pragma unroll
            for (int d = 1; d < 8; d <<= 1) {
#pragma unroll
                for (int k = 0; k < 3; k++) {
                    lo[k] = fminf(lo[k], __shfl_xor_sync(0xffffffffu, lo[k], d));
                    hi[k] = fmaxf(hi[k], __shfl_xor_sync(0xffffffffu, hi[k], d));
                }
                cnt += __shfl_xor_sync(0xffffffffu, cnt, d);
            }
            if ((lane & 7) == 0) {
                int cl = sc * NB_SUPER_SIZE + (e >> 3);
                bb_lo[cl] = make_float4(lo[0], lo[1], lo[2], (float)cnt);
                bb_hi[cl] = make_float4(hi[0], hi[1], hi[2], 0.f);
            }
#pragma unroll
            for (int k = 0; k < 3; k++) { slo[k] = fminf(slo[k], lo[k]); shi[k] = fmaxf(shi[k], hi[k]); }
        }
#pragma unroll
        for (int d = 8; d < 32; d <<= 1) {
#pragma unroll
            for (int k = 0; k < 3; k++) {
                slo[k] = fminf(slo[k], __shfl_xor_sync(0xffffffffu, slo[k], d));
                shi[k] = fmaxf(shi[k], __shfl_xor_sync(0xffffffffu, shi[k], d));
            }
        }
        if (lane == 0) {
            sbb_lo[sc] = make_float4(slo[0], slo[1], slo[2], (float)col);
            sbb_hi[sc] = make_float4(shi[0], shi[1], shi[2], 0.f);
        }
        __syncwarp();
    }
}

// Arrays are sized and kernels launched for nsc_max = natoms/64 + columns super-clusters, a bound the
// host knows without reading anything back; the super-clusters between the actual count and the
// bound are written as empty ones (no atoms, no bounding box: they are never listed).
__global__ void k_grid_tail(int nsc_max, const NbTotals* __restrict__ tot, int pad_type, float4* __restrict__ xq,
                            int* __restrict__ type_slot, int* __restrict__ atom_of_slot, float4* __restrict__ bb_lo,
                            float4* __restrict__ bb_hi, float4* __restrict__ sbb_lo, float4* __restrict__ sbb_hi,
                            float3 pad_base, float3 pad_step)
{
    const int slot = tot->nsc * NB_SC_ATOMS + blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= nsc_max * NB_SC_ATOMS) return;
    const int e = slot & 63, sc = slot >> 6;
    xq[slot] = make_float4(pad_base.x - pad_step.x * (float)e, pad_base.y - pad_step.y * (float)(sc & 63), pad_base.z, 0.f);
    type_slot[slot] = pad_type;
    atom_of_slot[slot] = -1;
    if ((e & 7) == 0) {
        bb_lo[slot >> 3] = make_float4(1e30f, 1e30f, 1e30f, 0.f);
        bb_hi[slot >> 3] = make_float4(-1e30f, -1e30f, -1e30f, 0.f);
    }
    if (e == 0) {
        sbb_lo[sc] = make_float4(1e30f, 1e30f, 1e30f, -1.f);
        sbb_hi[sc] = make_float4(-1e30f, -1e30f, -1e30f, 0.f);
    }
}

// (a1) refresh of the cluster-ordered coordinates from caller-order x with the stored image.
__global__ void k_refresh_xq(int n, const float* __restrict__ x, const float* __restrict__ q,
                             const char4* __restrict__ image, const int* __restrict__ slot_of_atom, float3 box,
                             float4* __restrict__ xq)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    char4 im = image[i];
    float4 v;
    v.x = __fmaf_rn(-(float)im.x, box.x, x[3 * i]);
    v.y = __fmaf_rn(-(float)im.y, box.y, x[3 * i + 1]);
    v.z = __fmaf_rn(-(float)im.z, box.z, x[3 * i + 2]);
    v.w = q[i];
    xq[slot_of_atom[i]] = v;
}

// (a1) device-pointer nb_put_atoms in ONE launch: copy the caller's x, q, type into the context
// (the next search reads them) and, when a grid exists, refresh the cluster-ordered coordinates.
__global__ void __launch_bounds__(256) k_put(int n, const float* __restrict__ x, const float* __restrict__ q,
                                             const int* __restrict__ type, float* __restrict__ cx, float* __restrict__ cq,
                                             int* __restrict__ ctype, const char4* __restrict__ image,
                                             const int* __restrict__ slot_of_atom, float3 box, float4* __restrict__ xq)
{
    nb_pdl_wait();
    nb_pdl_trigger();
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float px = x[3 * i], py = x[3 * i + 1], pz = x[3 * i + 2];
    cx[3 * i] = px; cx[3 * i + 1] = py; cx[3 * i + 2] = pz;
    float pq;
    if (q) { pq = q[i]; cq[i] = pq; } else pq = cq[i];   // NULL: unchanged since the previous call
    if (type) ctype[i] = type[i];
    if (xq) {
        const char4 im = image[i];
        xq[slot_of_atom[i]] = make_float4(__fmaf_rn(-(float)im.x, box.x, px), __fmaf_rn(-(float)im.y, box.y, py),
                                          __fmaf_rn(-(float)im.z, box.z, pz), pq);
    }
}

}  // namespace

const void* nbi_put_kernel() { return (const void*)k_put; }

int nbi_put_device(nb_ctx* c, const float* x, const float* q, const int32_t* type, bool refresh)
{
    int n = c->natoms;
    NB_CUDA(c, nb_launch_pdl(k_put, dim3((n + 255) / 256), dim3(256), 0, c->stream, n, x, q, type, c->x.p, c->q.p, c->type.p, c->image.p, c->slot_of_atom.p,
                                                  make_float3(c->box[0], c->box[1], c->box[2]), refresh ? c->xq.p : nullptr));
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}

int nbi_refresh_xq(nb_ctx* c)
{
    int n = c->natoms;
    k_refresh_xq<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->x.p, c->q.p, c->image.p, c->slot_of_atom.p,
                                                         make_float3(c->box[0], c->box[1], c->box[2]), c->xq.p);
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}

int nbi_grid(nb_ctx* c)
{
    const int n = c->natoms;
    cudaStream_t st = c->stream;
    const float* L = c->box;
    NbStageTimer tm(c, NB_T_GRID);
    // A10: column side ~ (64/rho)^(1/3) so that a super-cluster is roughly cubic.
    double vol = (double)L[0] * L[1] * L[2];
    double side = cbrt(NB_SC_ATOMS * vol / (double)n);
    c->ncx = (int)fmax(1.0, floor(L[0] / side + 0.5));
    c->ncy = (int)fmax(1.0, floor(L[1] / side + 0.5));
    c->ncol = c->ncx * c->ncy;
    c->inv_cx = (float)(c->ncx / (double)L[0]);
    c->inv_cy = (float)(c->ncy / (double)L[1]);
    // local / non-local split (nb_set_local): the non-local atoms get a column set of their own behind the local one
    c->nclass = c->nlocal < n ? 2 : 1;
    c->ncol_tot = c->ncol * c->nclass;
    // sum over columns of ceil(count/64) <= natoms/64 + columns: everything below is sized by this bound
    c->nsc_max = n / NB_SC_ATOMS + c->ncol_tot;
    c->nclusters_max = c->nsc_max * NB_SUPER_SIZE;
    c->nslots_max = c->nsc_max * NB_SC_ATOMS;
    NB_CUDA(c, c->col_count.ensure(c->ncol_tot + 1, st));
    NB_CUDA(c, c->col_atom_off.ensure(c->ncol_tot + 1, st));
    NB_CUDA(c, c->col_sc_off.ensure(c->ncol_tot + 1, st));
    NB_CUDA(c, c->atom_col.ensure(n, st));
    NB_CUDA(c, c->atom_rank.ensure(n, st));
    NB_CUDA(c, c->col_atoms.ensure(n, st));
    NB_CUDA(c, c->image.ensure(n, st));
    NB_CUDA(c, c->xw_atom.ensure(n, st));
    NB_CUDA(c, c->slot_of_atom.ensure(n, st));
    NB_CUDA(c, c->xq.ensure(c->nslots_max + NB_C * NB_NDUMMY, st));   // + dummy clusters (index >= nclusters_max), see below
    NB_CUDA(c, c->type_slot.ensure(c->nslots_max + NB_C * NB_NDUMMY, st));
    NB_CUDA(c, c->atom_of_slot.ensure(c->nslots_max, st));
    NB_CUDA(c, c->bb_lo.ensure(c->nclusters_max, st));
    NB_CUDA(c, c->bb_hi.ensure(c->nclusters_max, st));
    NB_CUDA(c, c->sbb_lo.ensure(c->nsc_max, st));
    NB_CUDA(c, c->sbb_hi.ensure(c->nsc_max, st));
    NB_CUDA(c, c->f4.ensure(c->nslots_max + NB_C * NB_NDUMMY, st));
    NB_CUDA(c, cudaMemsetAsync(c->f4.p, 0, sizeof(float4) * (c->nslots_max + NB_C * NB_NDUMMY), st));
    NB_CUDA(c, cudaMemsetAsync(c->col_count.p, 0, sizeof(int) * (c->ncol_tot + 1), st));
    float3 box = make_float3(L[0], L[1], L[2]);
    k_bin<<<(n + 255) / 256, 256, 0, st>>>(n, c->x.p, c->q.p, c->type.p, c->ntypes, box, c->ncx, c->ncy, c->inv_cx, c->inv_cy,
                                           c->nlocal, c->image.p, c->xw_atom.p, c->atom_col.p, c->atom_rank.p, c->col_count.p, c->tot_dev);
    NB_LAUNCH_CHECK(c);
    k_col_scan<<<1, 1024, 0, st>>>(c->ncol_tot, c->ncol, c->col_count.p, c->col_atom_off.p, c->col_sc_off.p, c->tot_dev);
    NB_LAUNCH_CHECK(c);
    k_col_scatter<<<(n + 255) / 256, 256, 0, st>>>(n, c->atom_col.p, c->atom_rank.p, c->col_atom_off.p,
                                                   c->col_atoms.p);
    NB_LAUNCH_CHECK(c);
    if (c->cold) {
        // no capacity known yet: read the largest column population back and size the in-shared-memory sort from it
        NB_CUDA(c, cudaMemcpyAsync(c->tot_host, c->tot_dev, sizeof(NbTotals), cudaMemcpyDeviceToHost, st));
        NB_CUDA(c, cudaStreamSynchronize(st));
        int want = c->tot_host->max_col + c->tot_host->max_col / 8 + 8, np2 = 64;
        while (np2 < want) np2 <<= 1;
        if (np2 / 2 >= c->tot_host->max_col + 8 && np2 > 64) np2 >>= 1;   // (head-room only where the power of two leaves some)
        c->np2_col = np2;
    }
    const int np2 = c->np2_col;
    size_t smem = (size_t)np2 * sizeof(unsigned long long);
    if (smem > 200 * 1024)
        return nb_fail(c, NB_ERR_OVERFLOW, "grid column holds %d atoms; the in-shared-memory z-sort takes at most 25600",
                       c->tot_host->max_col);
    NB_CUDA(c, cudaFuncSetAttribute(k_col_layout, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    float pb[3], pd[3];
    for (int k = 0; k < 3; k++) {
        pd[k] = (float)(L[k] / (floor(L[k] / 3.0) + 0.5));   // L/d half-integer, d in (2, 6] nm (2L for L < 3)
        pb[k] = (float)(-(2.0 * L[k] + 8.0));
    }
    k_col_layout<<<c->ncol_tot, 32 * NB_LAYOUT_WARPS, smem, st>>>(c->ncy, c->ncol, c->col_atom_off.p, c->col_sc_off.p, c->col_atoms.p,
                                             c->xw_atom.p, c->type.p, c->ntypes, np2, c->xq.p, c->type_slot.p,
                                             c->atom_of_slot.p, c->slot_of_atom.p, c->bb_lo.p, c->bb_hi.p,
                                             c->sbb_lo.p, c->sbb_hi.p, make_float3(pb[0], pb[1], pb[2]),
                                             make_float3(pd[0], pd[1], pd[2]), c->tot_dev);
    NB_LAUNCH_CHECK(c);
    k_grid_tail<<<(c->ncol_tot * NB_SC_ATOMS + 255) / 256, 256, 0, st>>>(c->nsc_max, c->tot_dev, c->ntypes, c->xq.p, c->type_slot.p,
                                                                   c->atom_of_slot.p, c->bb_lo.p, c->bb_hi.p, c->sbb_lo.p,
                                                                   c->sbb_hi.p, make_float3(pb[0], pb[1], pb[2]),
                                                                   make_float3(pd[0], pd[1], pd[2]));
    NB_LAUNCH_CHECK(c);
    if (c->dummy_at != (const void*)(c->xq.p + c->nslots_max) || c->dummy_box[0] != L[0] || c->dummy_box[1] != L[1] ||
        c->dummy_box[2] != L[2]) {
        // (rewritten only when the box or their place in the arrays has changed)
        // Dummy j-clusters (index nclusters_max .. nclusters_max + NB_NDUMMY - 1): padding-like atoms beyond the
        // padding lattice that interact with nothing.  The prune kernel may fill an inner list
        // segment up to a multiple of 32 atoms with them; the (zero) forces the force kernel adds to their
        // slots are never read, and spreading them over NB_NDUMMY clusters avoids atomic hot spots.
        std::vector<float4> hx((size_t)NB_C * NB_NDUMMY);
        std::vector<int32_t> ht((size_t)NB_C * NB_NDUMMY, c->ntypes);
        for (size_t i = 0; i < hx.size(); i++)
            hx[i] = make_float4(pb[0] - pd[0] * (float)(64 + (i % NB_C)), pb[1], pb[2], 0.f);
        NB_CUDA(c, cudaMemcpyAsync(c->xq.p + c->nslots_max, hx.data(), sizeof(float4) * hx.size(), cudaMemcpyHostToDevice, st));
        NB_CUDA(c, cudaMemcpyAsync(c->type_slot.p + c->nslots_max, ht.data(), sizeof(int32_t) * ht.size(), cudaMemcpyHostToDevice, st));
        NB_CUDA(c, cudaStreamSynchronize(st));
        c->dummy_at = c->xq.p + c->nslots_max;
        for (int k = 0; k < 3; k++) c->dummy_box[k] = L[k];
    }
    c->grid_box[0] = L[0];
    c->grid_box[1] = L[1];
    c->grid_box[2] = L[2];
    c->have_grid = true;
    c->st.ncolumns_x = c->ncx;
    c->st.ncolumns_y = c->ncy;
    c->st.cluster_size = NB_C;
    return NB_OK;
}
