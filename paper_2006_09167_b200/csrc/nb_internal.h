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
#define NB_NENT (2 * NB_NHALF)        // list elements per super-cluster: (j class, shift); element e of super-cluster sci
                                      // is sci * NB_NENT + jcls * NB_NHALF + h.  j class 1 = non-local j clusters
                                      // (nb_set_local; empty otherwise), so every element, work unit and segment is
                                      // purely local or non-local
#define NB_BATCH 32                   // joint j entries per mask word (one ballot)
#define NB_MAX_UNIT_BATCHES 16        // a work unit spans at most this many batches of one list element
#define NB_NDUMMY 1024                // dummy j-clusters behind the real ones (spread the never-read force adds)
#define NB_PAD_TYPE_ROW 1             // LJ table carries one extra all-zero type for padding atoms

// Counts produced on the device during a search.  Lives in device memory (`tot_dev`) where the stage
// kernels read their bounds from, and is copied to a pinned host mirror once, at the end of nb_search:
// the host sizes buffers from the previous search with head-room and only reads counts back to check
// that nothing overflowed ("host only reads back list counts when it must grow buffers").
struct NbTotals {
    int nsc, max_col;          // (a2) super-clusters, largest column population
    int njslots;               // (a3) joint j slots (multiple of NB_BATCH)
    int nunits;                // (a5) work units
    int nmask;                 // (a4) joint entries with an exclusion mask
    int il_total, ilm_total;   // extents of the compact lists (sum of segment capacities)
    int nseg_launch;           // segments with a non-empty outer list
    int overflow;              // NB_OVF_* bits: a stage found its buffer too small and did nothing
    int bad_type;              // an atom type outside [0, ntypes)
    int nsc_local;             // (a2) super-clusters of local atoms: they come first (nb_set_local; = nsc otherwise)
    int nseg_local;            // non-empty segments whose pairs are local-local: first in the force kernel's order
    int pad[4];
};
enum { NB_OVF_COL = 1, NB_OVF_JOINT = 2, NB_OVF_UNITS = 4, NB_OVF_MASKS = 8, NB_OVF_IL = 16, NB_OVF_ILM = 32 };
#define NB_SEG_MAXKEY 2080              // segment length key (see k_ilist_caps) is below this
#define NB_MAX_SORT_PARTS 16            // rolling parts whose prune order is sorted longest first (more: canonical order)

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
    float rcv2;           // rc_vdw^2 (twin cut-offs; = rc^2 otherwise)
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
    bool twin = false;                         // rc_vdw < rc: the TWIN kernel flavours

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
    // local / non-local split (nb_set_local): atoms [0, nlocal) are local, the rest non-local (halo).
    // The two classes are gridded into separate column sets (ncol_tot = nclass * ncol columns, class 1 after class 0),
    // so that clusters, super-clusters, list elements and segments are pure; nlocal = natoms: one class, nothing changes.
    int nlocal = 0, nclass = 1, ncol_tot = 0;
    int nsc_local = 0, nseg_local = 0;         // known after the end-of-search synchronisation
    cudaStream_t stream_hp = nullptr;          // high-priority stream of the non-local kernel
    cudaEvent_t ev_nl_in = nullptr, ev_nl_kernel = nullptr, ev_nl_done = nullptr;
    bool nl_pending = false;                   // nb_forces_nonlocal enqueued, nb_forces_local not yet
    double *nl_energies = nullptr, *nl_virial = nullptr;   // the caller's outputs of that pending pair of calls
    float inv_cx = 0.f, inv_cy = 0.f;          // columns per nm
    DevBuf<int32_t> col_count, col_atom_off, col_sc_off, atom_col, atom_rank, col_atoms;
    DevBuf<char4> image;                       // periodic image fixed at the last search
    DevBuf<float4> xw_atom;                    // wrapped (x,y,z,q) in caller order, search scratch
    int nsc = 0, nslots = 0, nclusters = 0, max_col_count = 0;   // exact, known after the end-of-search synchronisation
    int nclusters_max = 0, nslots_max = 0;     // nsc_max * 8, * 64: array extents; the dummy clusters start at nclusters_max
    DevBuf<float4> xq;                         // [nslots] x,y,z,q   (cluster order)
    DevBuf<int32_t> type_slot, atom_of_slot, slot_of_atom;
    DevBuf<float4> bb_lo, bb_hi;               // per cluster; lo.w = number of real atoms
    DevBuf<float4> sbb_lo, sbb_hi;             // per super-cluster
    DevBuf<float4> f4;                         // [nslots] force accumulator (x,y,z,unused), kept zero between calls

    // --- pair list (a3, a4) ---
    int nent = 0;                              // nsc * NB_NENT (super-cluster, j class, shift) slots, some empty
    DevBuf<int32_t> ent_count;                 // [nent] joint entries per slot
    DevBuf<int32_t> ent_jbegin;                // [nent+1] first j slot (multiple of NB_BATCH)
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

    // --- device-side counts (nb_list.cu) ---
    NbTotals* tot_dev = nullptr;               // device
    NbTotals* tot_host = nullptr;              // pinned mirror, valid after the end-of-search synchronisation
    int nsm = 148;                             // multiprocessors of the device (persistent kernels are sized by it)
    bool cold = true;                          // no capacities known yet (first search, or after an overflow): stage by stage
    int nsc_max = 0;                           // natoms/64 + columns: host-side bound of nsc, everything is sized and launched by it
    int np2_col = 0;                           // shared-memory sort size of k_col_layout (power of two >= largest column, with head-room)
    size_t cap_jslots = 0, cap_units = 0, cap_masks = 0, cap_il = 0, cap_ilm = 0;   // what the list buffers hold
    bool stats_dirty = true;                   // list statistics are computed lazily in nb_get_stats
    bool planes_dirty = false;                 // plane_inner (introspection only) is stale with respect to the compact inner list

    // --- work units (a5) ---
    DevBuf<int4> units_canon;                  // {entry slot, batch begin, batch end, sci}, canonical order (rolling parts are ranges of it)
    DevBuf<int32_t> unit_nsplit, unit_off;     // [nent] scan scratch
    int nunits = 0;
    // prune launch order per nparts: segment ids (positions in the force kernel's order), each rolling part
    // longest list first; one cached table per recently used nparts, rebuilt lazily after a search
    struct PruneOrder { int nparts = 0; int64_t search = -1; DevBuf<int32_t> d; };
    PruneOrder prune_orders[4];
    int prune_order_next = 0;
    DevBuf<int32_t> sort_hist;                 // [parts * NB_SEG_MAXKEY] counting-sort buckets
    DevBuf<int32_t> seg_len;                   // [nunits*8] by s0: sort key of the launch orders (outer list length)
    float dummy_box[3] = {0, 0, 0};            // box the dummy clusters were last written for
    const void* dummy_at = nullptr;            // ... and where

    // --- compact lists (a3 -> a6 -> a7), per (work unit, i-cluster) SEGMENT ---
    // s0 = canonical unit * 8 + i-cluster names a segment at search time; t = its position in the force
    // kernel's launch order (longest outer list first) names it everywhere afterwards.
    DevBuf<int32_t> il_off, ilm_off;           // [nunits*8] by s0: first entry of the segment in il / ilm (scan output)
    DevBuf<int32_t> seg_of_s0;                 // [nunits*8] s0 -> t
    DevBuf<int4> segd;                         // [nunits*8] by t: {il offset, ilm offset, i-cluster | shift id << 26, canonical unit}
    DevBuf<int2> ol_cnt;                       // [nunits*8] by t: OUTER {cluster pairs without a mask, with a mask}
    DevBuf<int2> seg_cnt[2];                   // [nunits*8] by t: INNER {j-atom entries (multiple of 32), masked cluster pairs}
    DevBuf<int32_t> olu;                       // OUTER list, cluster pairs without a mask: cj, segment at il offset; written once per search
    DevBuf<int2> olm;                          // OUTER list, cluster pairs with a mask: {cj, mask ref}, segment at ilm offset
    DevBuf<int32_t> il[2];                     // INNER list: slots of the surviving j atoms (+ dummies up to a multiple of 32)
    DevBuf<int2> ilm[2];                       // INNER list: surviving masked cluster pairs {cj, mask ref}
    // Two inner buffers: nb_prune_overlapped writes the part it prunes into the buffer the force kernel is
    // NOT reading and the part flips at the next nb_put_atoms.  Bit p of bufmask = buffer holding part p
    // (parts as in buf_nparts); 0 everywhere unless the overlapped mode is in use.
    unsigned bufmask = 0;
    int buf_nparts = 1;
    int seg_part_nparts = 0;
    int64_t seg_part_search = -1;              // what seg_part was last computed for
    DevBuf<int32_t> seg_part;                  // [nunits*8] by t: rolling part of the segment under buf_nparts (read only while bufmask != 0)
    bool have_buf1 = false;
    int pending_part = -1;                     // overlapped prune in flight on side_stream (its part), else -1
    cudaStream_t side_stream = nullptr;
    cudaEvent_t ev_main = nullptr, ev_side = nullptr;
    size_t il_total = 0, ilm_total = 0;        // extents of il / ilm in use
    int nseg_launch = 0;                       // segments with a non-empty outer list (= force kernel grid)
    DevBuf<float4> ljrow;                      // [nclusters_max * 4 * (ntypes+1)] paired LJ rows per i-cluster (nb_force.cu), written at search
    DevBuf<double> fshift;                     // [27*3] per-shift i-force sums (virial)
    void* static_scratch = nullptr;            // nb_forces_static: device address of nb_force.cu's static scratch array on this
                                               // context's device (cudaGetSymbolAddress at nb_init), nullptr if that failed
    int static_scratch_cuda_err = 0;           // the cudaError_t of that failure

    // --- nb_step: the inner step (put + rolling prune + forces) as one CUDA graph launch ---
    // One cached graph per (part, nparts, rlist_inner); captured on a private stream (the caller's may be the legacy
    // default stream, which cannot be captured) the second time a key is used after a search, updated in place after
    // the next search; the caller's x and f pointers are patched into the put / gather nodes at every launch.
    struct StepGraph {
        int part = -1, nparts = 0;
        float rl = 0.f;
        int64_t warm_search = -1;              // the plain path ran for this key on this list (buffers, orders, tables exist)
        int64_t graph_search = -1;             // the graph was captured for this list
        cudaGraph_t graph = nullptr;
        cudaGraphExec_t exec = nullptr;
        cudaGraphNode_t put = nullptr, gather = nullptr;
        bool broken = false;                   // capture or instantiation failed: always the plain path
    };
    StepGraph step_graphs[8];
    int step_graph_next = 0;
    cudaStream_t capture_stream = nullptr;

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
// The compact inner list is kept at single-j-ATOM granularity (reading A22): an unmasked entry is the slot index of one
// j atom, listed for the i-cluster iff it is within rlist_inner of one of the cluster's atoms.  Against whole j-clusters
// that skips 35 % of the atom-pair slots on the water boxes (25 % against half j-clusters, the paper's 8x4 shape): the
// lanes of the force kernel own one j atom each anyway, so the finer list costs nothing there; it is four times the
// entries of a half-cluster list (4 B per listed j atom).  Cluster pairs that carry a mask stay whole: {cj, mask ref}.
//
// Closes a segment of nu unmasked atom entries + nm masked cluster pairs (one warp): the unmasked count is filled up to
// a multiple of 32 (one force-kernel step = 32 j atoms) with dummy atoms (far from everything, nb_grid.cu).
__device__ __forceinline__ void nb_ilist_finish(int nu, int nm, int salt, int lane, int cj_dummy,
                                                int32_t* __restrict__ il, int2* __restrict__ ilm, int2* __restrict__ cnt)
{
    const int rem = nu & 31;
    if (rem != 0) {
        if (lane < 32 - rem) il[nu + lane] = 8 * cj_dummy + ((salt + lane) & (8 * NB_NDUMMY - 1));
        nu += 32 - rem;
    }
    if (lane == 0) *cnt = make_int2(nu, nm);
}

// Rolling part of a canonical work unit: part p of k is the range [p*nu/k, (p+1)*nu/k) (reading A15).
__host__ __device__ __forceinline__ int nb_part_of_unit(int u, int nparts, int nunits)
{
    if (nparts <= 1) return 0;
    int p = (int)(((long long)u * nparts) / nunits);
    if (p > nparts - 1) p = nparts - 1;
    while (p + 1 < nparts && ((long long)(p + 1) * nunits) / nparts <= u) p++;
    while (p > 0 && ((long long)p * nunits) / nparts > u) p--;
    return p;
}
// Which of the two inner-list buffers holds the segment of canonical unit u (nb_ctx::bufmask).
__device__ __forceinline__ int nb_seg_buf(int u, unsigned bufmask, int nparts, int nunits)
{
    return bufmask ? (int)((bufmask >> nb_part_of_unit(u, nparts, nunits)) & 1u) : 0;
}
#endif

// Programmatic dependent launch: a kernel launched with nb_launch_pdl may be scheduled while its predecessor in the
// stream is still draining (its launch latency and the predecessor's tail overlap); it must call nb_pdl_wait() before it
// touches anything -- the wait returns when the predecessor grid has completed and its writes are visible.  A kernel calls
// nb_pdl_trigger() to let its successor start being scheduled (all blocks must have called it or exited).
#ifdef __CUDACC__
__device__ __forceinline__ void nb_pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void nb_pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <typename... KArgs, typename... Args>
inline cudaError_t nb_launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
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
int nbi_forces(nb_ctx* c, float* f, double* energies, double* virial, float rlist_inner_fused = 0.f);   // (a7)-(a8) nb_force.cu
int nbi_list_count(nb_ctx* c, int which, int64_t* n);      // nb_list.cu
int nbi_list_dump(nb_ctx* c, int which, int32_t* ci, int32_t* cj, int32_t* shift, uint64_t* pairmask,
                  int32_t* part);
int nbi_measure_fp32_peak(nb_ctx* c, double* fma_per_s);   // nb_force.cu
int nbi_measure_fp32_pipe(nb_ctx* c, double* cycles);       // nb_force.cu
int nbi_count_pairs(nb_ctx* c, int64_t* n_interacting, int64_t* n_excluded);   // nb_force.cu
int nbi_count_slots(nb_ctx* c, int64_t* slots);            // nb_force.cu
int nbi_inner_dump(nb_ctx* c, int64_t* n, int32_t* ci, int32_t* entry, int32_t* shift, int32_t* kind, int32_t* part);   // nb_force.cu
int nbi_prune_overlapped(nb_ctx* c, float rlist_inner, int part, int nparts);   // nb_prune.cu
int nbi_commit_pending(nb_ctx* c);                          // nb_prune.cu: join an overlapped prune and flip its part
int nbi_prepare_parts(nb_ctx* c, int nparts);               // nb_prune.cu: part table and prune launch order for nparts, now
int nbi_consolidate(nb_ctx* c);                             // nb_prune.cu: move every segment back to inner buffer 0
int nbi_rebuild_inner_planes(nb_ctx* c);                    // nb_list.cu: plane_inner from the compact inner list (introspection)
int nbi_list_stats(nb_ctx* c);                              // nb_list.cu: lazily computed list statistics
int nbi_prune_order(nb_ctx* c, int nparts, const int32_t** table);   // nb_list.cu: prune launch order for nparts rolling parts
int nbi_ljrows(nb_ctx* c);                                  // nb_force.cu: paired LJ rows per i-cluster, at search time
int nbi_exclusive_scan(nb_ctx* c, const int32_t* in, int32_t* out, int64_t n, int32_t* total_dev);  // nb_list.cu
const void* nbi_put_kernel();                               // nb_grid.cu: the k_put entry (node lookup in captured graphs)
const void* nbi_gather4_kernel();                           // nb_force.cu: the k_gather4 entry
int nbi_split_setup(nb_ctx* c);                             // nb_force.cu: high-priority stream and events of the local / non-local split
void nbi_split_free(nb_ctx* c);
int nbi_forces_nonlocal(nb_ctx* c, float* f, double* energies, double* virial);               // nb_force.cu: non-local kernel + gather of the non-local atoms
int nbi_forces_local(nb_ctx* c, float* f);                  // nb_force.cu: local kernel + gather of the local atoms
int nbi_sync_nonlocal(nb_ctx* c);
void nbi_static_scratch_setup(nb_ctx* c);                   // nb_force.cu: resolves c->static_scratch (the context's device is current)
int nbi_forces_static(nb_ctx* c, float* f, double* energies, double* virial);   // nb_force.cu: nb_forces_static
