// nb_internal.h -- context and device data layout of the B200 cluster-pair library.
// Not part of the public ABI (include/nb.h is).  Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "../../include/nb.h"

#define NB_C NB_CLUSTER_SIZE          // atoms per cluster
#define NB_SC_ATOMS 64                // atoms per super-cluster (8 clusters x 8 atoms)
#define NB_NHALF 14                   // zero shift + 13 shifts with s >lex 0
#define NB_BATCH 32                   // joint j entries per mask word (one ballot)
#define NB_MAX_UNIT_BATCHES 16        // a work unit spans at most this many batches of one list element
#define NB_NDUMMY 1024                // dummy j-clusters behind the real ones (spread the never-read force adds)
#define NB_PAD_TYPE_ROW 1             // LJ table carries one extra all-zero type for padding atoms

// One growable device array.
template <typename T>
struct DevBuf {
    T* p = nullptr;
    size_t cap = 0;
    cudaError_t ensure(size_t n, cudaStream_t st, bool keep = false)
    {
        if (n <= cap) return cudaSuccess;
        size_t ncap = n + n / 4 + 64;
        T* np_ = nullptr;
        cudaError_t e = cudaMalloc((void**)&np_, ncap * sizeof(T));
        if (e != cudaSuccess) return e;
        if (p) {
            if (keep && cap) {
                e = cudaMemcpyAsync(np_, p, cap * sizeof(T), cudaMemcpyDeviceToDevice, st);
                if (e != cudaSuccess) return e;
            }
            cudaStreamSynchronize(st);
            cudaFree(p);
        }
        p = np_;
        cap = ncap;
        return cudaSuccess;
    }
    void release()
    {
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
    }
};

// Parameters every kernel needs, passed by value.
struct NbConst {
    float box[3];
    float rc2;            // rc^2
    float epsfac;
    float beta, beta2, beta3;
    float ewald_shift;    // erfc(beta rc)/rc if potential-shift else 0
    float two_krf, krf, crf;
    float lj_sh6, lj_sh12;  // rc^-6, rc^-12 if potential-shift else 0
    int ntypes1;          // ntypes + 1 (row length of the padded LJ table)
    // Ewald correction fit as polynomials in r^2 (beta folded in), every coefficient duplicated
    // for the packed FFMA2 form: ewp2[k] = beta^(3+2k) P_k, ewq2[k] = beta^(2k) Q_k.
    float2 ewp2[5], ewq2[6];
};

struct nb_ctx {
    nb_params prm;
    cudaStream_t stream = nullptr;
    char err[512];
    int natoms = 0, ntypes = 0;
    NbConst kc;
    float beta = 0.f;
    double beta_d = 0.0;                       // Ewald beta in fp64 (coefficient folding)

    // --- state machine ---
    bool have_atoms = false, have_grid = false, have_list = false, atoms_since_search = false;
    float box[3] = {0, 0, 0};
    float grid_box[3] = {0, 0, 0};
    float rlist_outer = 0.f;
    int last_nparts = 1;

    // --- caller-order copies (a1) ---
    DevBuf<float> x, q;
    DevBuf<int32_t> type;
    DevBuf<float> stage_x, stage_q, stage_f;   // staging for the _host entry points
    DevBuf<int32_t> stage_type;
    DevBuf<double> stage_ev;

    // --- topology ---
    DevBuf<int32_t> excl_off, excl_idx;
    int64_t nexcl = 0;
    DevBuf<float2> ljtab;        // [(ntypes+1)^2] (6*c6, 12*c12); last row/column zero

    // --- grid (a2) ---
    int ncx = 0, ncy = 0, ncol = 0;
    float inv_cx = 0.f, inv_cy = 0.f;          // columns per nm
    DevBuf<int32_t> col_count, col_atom_off, col_sc_off, atom_col, atom_rank, col_atoms;
    DevBuf<int32_t> grid_totals;               // [4]: nsc, max column count, ...
    DevBuf<char4> image;                       // periodic image fixed at the last search
    DevBuf<float4> xw_atom;                    // wrapped (x,y,z,q) in caller order, search scratch
    int nsc = 0, nslots = 0, nclusters = 0, max_col_count = 0;
    DevBuf<float4> xq;                         // [nslots] x,y,z,q   (cluster order)
    DevBuf<int32_t> type_slot, atom_of_slot, slot_of_atom;
    DevBuf<float4> bb_lo, bb_hi;               // per cluster; lo.w = number of real atoms
    DevBuf<float4> sbb_lo, sbb_hi;             // per super-cluster
    DevBuf<float4> f4;                         // [nslots] force accumulator (x,y,z,unused), kept zero between calls

    // --- pair list (a3, a4) ---
    int nent = 0;                              // nsc * NB_NHALF (super-cluster, shift) slots, some empty
    DevBuf<int32_t> ent_count;                 // [nent] joint entries per slot
    DevBuf<int32_t> ent_jbegin;                // [nent+1] first j slot (multiple of NB_BATCH)
    std::vector<int32_t> h_ent_count, h_ent_jbegin;
    int64_t njslots = 0, nbatch = 0;
    DevBuf<int2> jl;                           // [njslots] {cj, exclusion mask ref (0 = none)}
    DevBuf<uint8_t> imask_outer;               // [njslots] 8-bit interaction mask
    DevBuf<uint32_t> plane_outer, plane_inner; // [nbatch*8] bit-planes of the masks, word = (batch, i-cluster)
    DevBuf<uint32_t> plane_excl;               // [nbatch*8] bit set: the entry's exclusion mask is non-trivial for this i-cluster
    DevBuf<int32_t> batch_ent;                 // [nbatch] owning (super-cluster, shift) slot
    DevBuf<int32_t> scan_tmp, scan_blk;        // scratch for device scans
    DevBuf<unsigned long long> excl_masks;     // [(nmask+1)*8*2] {interact, count} per (ref, i-cluster)
    int64_t nmask = 0;
    DevBuf<long long> counters;                // device counters (list statistics)

    // --- work units (a5) ---
    std::vector<int4> h_units;
    DevBuf<int4> units_canon, units_sorted;    // {entry slot, batch begin, batch end, sci}
    DevBuf<int32_t> unit_order;                // canonical unit index, longest first (force kernel launch order)
    // prune launch order: (canonical unit*8 + i-cluster), each rolling part longest list first; one
    // cached table per recently used nparts, rebuilt lazily after a search
    struct PruneOrder { int nparts = 0; int64_t search = -1; DevBuf<int32_t> d; std::vector<int32_t> h; };
    PruneOrder prune_orders[4];
    int prune_order_next = 0;
    std::vector<int32_t> h_unit_order, h_seg_sorted, h_seg_pos;   // host copies made at search time (sources of async uploads)
    float dummy_box[3] = {0, 0, 0};            // box the dummy clusters were last written for
    const void* dummy_at = nullptr;            // ... and where
    int nunits = 0;

    // --- compact inner list (a6 -> a7): per (work unit, i-cluster) the j-clusters whose inner mask bit is set ---
    DevBuf<int32_t> il_off, ilm_off;           // [nunits*8] scan scratch: first entry of the segment in il / ilm
    DevBuf<int4> seg;                          // [nunits*8], one per (work unit, i-cluster), longest outer list first:
                                               // {il offset, ilm offset, unmasked half-cluster entries (multiple of 8), masked entries}
    DevBuf<int32_t> unit_pos;                  // canonical unit index -> launch position (inverse of unit_order)
    DevBuf<int32_t> seg_pos;                   // [nunits*8] (unit launch position*8 + i-cluster) -> index into seg (longest first)
    DevBuf<int2> seg_ci;                       // [nunits*8] {i-cluster, shift id} of each seg entry
    size_t il_total = 0, ilm_total = 0;        // allocated extents of il / ilm in use (sum of segment capacities)
    int nseg_launch = 0;                       // seg entries with a non-empty outer list (= force kernel grid)
    std::vector<int32_t> h_caps;               // host scratch
    DevBuf<int32_t> il;                        // cj of cluster pairs without a mask for this i-cluster
    DevBuf<int2> ilm;                          // {cj, mask ref} of cluster pairs with a mask, plus each segment's tail
    // compact OUTER list (a3 -> a6): what the prune kernel streams; written once per search
    DevBuf<int2> ol;                           // {cj, unit-local joint slot}; segment at il offset + ilm offset: the cluster pairs
                                               // without a mask, then (from a multiple of 4 on) those with a mask
    DevBuf<int2> ol_cnt;                       // [nunits*8] {unmasked, masked} entries per segment (index: unit launch position*8 + i-cluster)
    DevBuf<double> fshift;                     // [27*3] per-shift i-force sums (virial)

    // --- per-stage device timing (nb_timing_enable / nb_timing_read) ---
    bool timing = false;
    unsigned timing_mask = ~0u;                // stages to time (nb_timing_stages)
    struct TimRec { int kind; cudaEvent_t e0, e1; };
    std::vector<TimRec> tim_open;              // recorded, not yet read
    std::vector<cudaEvent_t> tim_pool;         // recycled events
    double tim_ms[NB_T_NKINDS] = {0};
    int64_t tim_n[NB_T_NKINDS] = {0};

    nb_stats st;
};

// RAII stage timer: CUDA events on the context's stream around the launches of one stage.
// Costs nothing unless nb_timing_enable(ctx, 1) was called.
struct NbStageTimer {
    nb_ctx* c;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int kind;
    static cudaEvent_t get(nb_ctx* c)
    {
        if (!c->tim_pool.empty()) { cudaEvent_t e = c->tim_pool.back(); c->tim_pool.pop_back(); return e; }
        cudaEvent_t e = nullptr;
        cudaEventCreate(&e);
        return e;
    }
    NbStageTimer(nb_ctx* c_, int kind_) : c(c_), kind(kind_)
    {
        if (!c->timing || !((c->timing_mask >> kind_) & 1u)) return;
        e0 = get(c);
        e1 = get(c);
        cudaEventRecord(e0, c->stream);
    }
    ~NbStageTimer()
    {
        if (!e0) return;
        cudaEventRecord(e1, c->stream);
        c->tim_open.push_back({kind, e0, e1});
    }
};

// Half-set of shifts: index 0 is the zero shift, 1..13 are the shifts with s >lex 0 in
// (sx,sy,sz) order (reading A14).  Decoded with nb_shift_vec().
__host__ __device__ inline int nb_half_shift_id(int h)
{
    // ids = (sx+1) + 3*(sy+1) + 9*(sz+1)
    const int ids[NB_NHALF] = {13, /* sx=+1: all (sy,sz) */ 2, 5, 8, 11, 14, 17, 20, 23, 26,
                               /* sx=0, sy=+1 */ 7, 16, 25, /* sx=sy=0, sz=+1 */ 22};
    return ids[h];
}
__host__ __device__ inline void nb_shift_vec(int id, int& sx, int& sy, int& sz)
{
    sx = id % 3 - 1;
    sy = (id / 3) % 3 - 1;
    sz = id / 9 - 1;
}

int nb_fail(nb_ctx* c, int code, const char* fmt, ...);

#ifdef __CUDACC__
// The compact inner list is kept at HALF j-cluster granularity (4 atoms): an unmasked entry is the
// half-cluster index hc = 2*cj + half, whose atoms are the slots 4*hc .. 4*hc+3.  The prune kernel
// keeps a half iff one of its atoms is within rlist_inner of the i-cluster, which skips about a
// tenth of the atom-pair slots a whole-cluster list evaluates (the cluster-pair "split" of the
// paper's GPU lists).  Masked entries {cj, mask ref} stay whole clusters.
//
// Closes a segment of nu unmasked half entries + nm masked entries (one warp): the unmasked count
// is filled up to a multiple of 8 (one force-kernel step = 8 half-clusters) with dummy half-clusters.
__device__ __forceinline__ void nb_ilist_finish(int nu, int nm, int salt, int lane, int cj_dummy,
                                                int32_t* __restrict__ il, int2* __restrict__ ilm, int2* __restrict__ cnt)
{
    const int rem = nu & 7;
    if (rem != 0) {
        if (lane < 8 - rem) il[nu + lane] = 2 * cj_dummy + ((salt + lane) & (2 * NB_NDUMMY - 1));
        nu += 8 - rem;
    }
    if (lane == 0) *cnt = make_int2(nu, nm);
}

// Writes the compact inner list segment of (unit, i-cluster warp) from the unit's inner mask
// words `bits_of(b)` (b = batch index relative to the unit), keeping BOTH halves of every
// cluster (used after a search: inner := outer).  Entries whose exclusion mask is trivial for
// this i-cluster go to `il` (two half-cluster indices), the others to `ilm` {cj, mask ref}.
// One warp, all 32 lanes.
template <typename BitsOf>
__device__ __forceinline__ void nb_ilist_write(BitsOf bits_of, int b0, int b1, int warp, int lane, int cj_dummy,
                                               const uint32_t* __restrict__ plane_excl, const int2* __restrict__ jl,
                                               int32_t* __restrict__ il, int2* __restrict__ ilm, int2* __restrict__ cnt)
{
    const unsigned lt = (1u << lane) - 1u;
    int nu = 0, nm = 0;
    for (int b = b0; b < b1; b++) {
        const unsigned bits = bits_of(b - b0);
        const unsigned eb = plane_excl[(size_t)b * 8 + warp] & bits, nb = bits & ~eb;
        if ((bits >> lane) & 1u) {
            const int2 e = jl[(size_t)b * 32 + lane];
            if ((nb >> lane) & 1u)
                *reinterpret_cast<int2*>(&il[nu + 2 * __popc(nb & lt)]) = make_int2(2 * e.x, 2 * e.x + 1);
            else ilm[nm + __popc(eb & lt)] = e;
        }
        nu += 2 * __popc(nb);
        nm += __popc(eb);
    }
    __syncwarp();
    nb_ilist_finish(nu, nm, b0 * 8 + warp, lane, cj_dummy, il, ilm, cnt);
}
#endif

#define NB_CUDA(c, expr)                                                                              \
    do {                                                                                              \
        cudaError_t e__ = (expr);                                                                     \
        if (e__ != cudaSuccess)                                                                       \
            return nb_fail((c), e__ == cudaErrorMemoryAllocation ? NB_ERR_NOMEM : NB_ERR_CUDA,        \
                           "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
    } while (0)

#define NB_LAUNCH_CHECK(c)                                                                            \
    do {                                                                                              \
        (c)->st.kernel_launches++;                                                                    \
        NB_CUDA((c), cudaGetLastError());                                                             \
    } while (0)

// Stage implementations (one translation unit each).
int nbi_grid(nb_ctx* c);                                   // (a2) nb_grid.cu
int nbi_refresh_xq(nb_ctx* c);                             // (a1) nb_grid.cu
int nbi_put_device(nb_ctx* c, const float* x, const float* q, const int32_t* type, bool refresh);   // (a1) nb_grid.cu
int nbi_search(nb_ctx* c, float rlist);                    // (a3)-(a5) nb_list.cu
int nbi_prune(nb_ctx* c, float rlist_inner, int part, int nparts);   // (a6) nb_prune.cu
int nbi_forces(nb_ctx* c, float* f, double* energies, double* virial);   // (a7)-(a8) nb_force.cu
int nbi_list_count(nb_ctx* c, int which, int64_t* n);      // nb_list.cu
int nbi_list_dump(nb_ctx* c, int which, int32_t* ci, int32_t* cj, int32_t* shift, uint64_t* pairmask,
                  int32_t* part);
int nbi_measure_fp32_peak(nb_ctx* c, double* fma_per_s);   // nb_force.cu
int nbi_count_pairs(nb_ctx* c, int64_t* n_interacting, int64_t* n_excluded);   // nb_force.cu
int nbi_count_slots(nb_ctx* c, int64_t* slots);            // nb_force.cu
int nbi_inner_dump(nb_ctx* c, int64_t* n, int32_t* ci, int32_t* entry, int32_t* shift, int32_t* kind);   // nb_force.cu
int nbi_exclusive_scan(nb_ctx* c, const int32_t* in, int32_t* out, int64_t n, int32_t* total_dev);  // nb_list.cu
