/*
 * nb.h -- C ABI of the B200 cluster-pair short-range non-bonded library.
 *
 * The five working calls are the ones BASELINE.json's north_star lists
 * (nb_init / nb_put_atoms / nb_search / nb_prune / nb_forces); they follow the paper's
 * statement of the problem: positions go in and forces come out every step
 * (PAPER.md L105), the pair list is built rarely and reused for many steps (L185, L193),
 * pruning runs in rolling chunks between force computations (L193).
 *
 * Conventions
 *  - Pointers marked [dev] are CUDA device pointers owned by the caller; the library
 *    never frees them and never keeps them past the call.  Everything else is host memory.
 *    [host] variants (suffix _host) take plain host pointers and do the copies themselves.
 *  - Every call returns NB_OK or a negative NB_ERR_* code; nothing throws or exits.
 *    nb_last_error() gives a message for the last failure on that context.
 *  - All work is enqueued on the stream given in nb_params and returns without
 *    synchronising, except nb_search (one synchronisation at its end to read the list sizes
 *    back) and the introspection / _host calls.  Every call switches to the context's device
 *    and restores the caller's current device before returning.
 *  - Call order: nb_init -> nb_put_atoms -> nb_search -> { nb_put_atoms -> [nb_prune | nb_prune_overlapped]
 *    -> nb_forces }* -> nb_put_atoms -> nb_search ...; violations return NB_ERR_STATE.  The first use of a
 *    fresh list may be nb_forces_prune instead of nb_prune + nb_forces; nb_step / nb_step_host are one pass
 *    of the braces in one call; nb_forces_nonlocal + nb_forces_local (after nb_set_local and a search) or
 *    nb_forces_static stand where nb_forces does.
 *  - Units: nm, kJ/mol, e.  Rectangular periodic boxes only.  natoms, types, charges'
 *    layout and exclusions are fixed for the lifetime of a context (only
 *    positions change per step).
 *  - Between searches the caller passes CONTINUOUS (not re-wrapped) coordinates; the
 *    library applies the periodic image fixed for each atom at the last search.
 *
 * Cluster geometry: clusters of NB_CLUSTER_SIZE = 8 atoms, 8 clusters
 * (2x2x2 cells of the search grid) per super-cluster, one joint j-cluster list per
 * (super-cluster, periodic shift) with an 8-bit interaction mask per j-cluster.
 */
#ifndef NB_B200_H
#define NB_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NB_CLUSTER_SIZE 8
#define NB_SUPER_SIZE 8        /* clusters per super-cluster */
#define NB_NSHIFT 27
#define NB_SHIFT_CENTER 13     /* shift id = (sx+1) + 3*(sy+1) + 9*(sz+1), s in {-1,0,1}^3 */
#define NB_MAX_TYPES 96

typedef struct nb_ctx nb_ctx; /* opaque, owned by the library */

enum { NB_OK = 0, NB_ERR_ARG = -1, NB_ERR_STATE = -2, NB_ERR_CUTOFF = -3, NB_ERR_BOX = -4,
       NB_ERR_NOMEM = -5, NB_ERR_CUDA = -6, NB_ERR_OVERFLOW = -7 };
enum { NB_COUL_EWALD = 0, NB_COUL_RF = 1,
       NB_COUL_NONE = 2 /* LJ-only flavour (Fig. 6 workload): charges are ignored, E_coul = 0 */ };
enum { NB_MOD_NONE = 0, NB_MOD_POTSHIFT = 1 };

typedef struct {
    int32_t natoms, ntypes;          /* ntypes <= NB_MAX_TYPES */
    const float* lj_c6c12;           /* host [ntypes*ntypes*2]: c6 = 4 eps sigma^6, c12 = 4 eps sigma^12; copied */
    const int32_t* excl_off;         /* host CSR [natoms+1]; copied.  NULL = no exclusions */
    const int32_t* excl_idx;         /* host [excl_off[natoms]]; symmetric, no self entries; copied */
    float rc;                        /* interaction cut-off, nm (LJ and Coulomb; interact iff r^2 < rc^2) */
    int32_t coulomb;                 /* NB_COUL_* */
    float ewald_beta;                /* nm^-1; if <= 0 derived from ewald_rtol: erfc(beta*rc) = rtol.
                                        (beta*rc)^2 must be <= 12 (range of the correction fit) */
    float ewald_rtol;
    float eps_rf;                    /* reaction-field dielectric; <= 0 or inf -> infinity (eps_r = 1) */
    float epsfac;                    /* 1/(4 pi eps0); 0 -> 138.935458 kJ mol^-1 nm e^-2 */
    int32_t lj_modifier;             /* NB_MOD_*: potential-shift changes energies only */
    int32_t coul_modifier;           /* Ewald only; reaction-field always carries its own constant c_rf */
    int32_t device;                  /* CUDA ordinal */
    void* stream;                    /* cudaStream_t (NULL = legacy default stream) */
    float rc_vdw;                    /* twin cut-offs (PME load balancing scales only the electrostatics
                                        cut-off): LJ interacts iff r^2 < rc_vdw^2 and its potential shift is taken at rc_vdw;
                                        0 -> rc (single cut-off); otherwise 0 < rc_vdw <= rc */
} nb_params;

/* Counters for the last calls; all device work they describe has completed when
 * nb_get_stats returns (it synchronises the stream). */
typedef struct {
    int32_t cluster_size, nclusters, nsuper, nslots;
    int32_t ncolumns_x, ncolumns_y;
    int64_t n_sci_entries;           /* non-empty (super-cluster, shift) list elements */
    int64_t n_joint_outer;           /* joint j entries with any outer mask bit */
    int64_t n_pairs_outer;           /* listed cluster pairs (ci,cj,s): outer mask bits set */
    int64_t n_pairs_inner;           /* cluster pairs with the inner mask bit set (after pruning) */
    int64_t n_excl_masks;            /* joint entries carrying a non-trivial exclusion mask */
    int64_t n_work_units;            /* list chunks scheduled by the force/prune kernels (L199-L201) */
    int64_t slots_last_forces;       /* atom-pair slots the force kernel evaluates over the current inner list (= nb_count_slots):
                                        8 per listed j atom (x 8 i atoms), 64 per masked cluster pair; 0 before the first nb_forces */
    int64_t kernel_launches;         /* kernels launched by this context so far */
    int64_t search_count, prune_count, force_count;
    int32_t list_grow_retries;       /* searches repeated because a list buffer sized from the previous search was too small */
    float ewald_beta;
} nb_stats;

/* Creates a context.  Copies the LJ table and exclusions.  NB_ERR_ARG on bad sizes,
 * an exclusion index out of range, a self entry or an entry (i,j) without its mirror (j,i),
 * rc <= 0, or (beta*rc)^2 > 12. */
int nb_init(const nb_params* p, nb_ctx** out);

/* (a1) Coordinate staging.  x [dev] natoms*3 fp32, q [dev] natoms,
 * type [dev] natoms (0 <= type < ntypes), box host [3] (Lx,Ly,Lz > 0).  Copies them; if a
 * grid exists and the box is unchanged, also refreshes the cluster-ordered (x,y,z,q) array.
 * q and/or type may be NULL after the first call: "unchanged since the previous nb_put_atoms"
 * (only positions change from step to step); NB_ERR_ARG on the first call. */
int nb_put_atoms(nb_ctx*, const float* x, const float* q, const int32_t* type, const float box[3]);
/* Same with host pointers (pageable or pinned); copies are enqueued on the stream. */
int nb_put_atoms_host(nb_ctx*, const float* x, const float* q, const int32_t* type, const float box[3]);

/* (a2)-(a5) Gridding into clusters (L129-L131), bounding-box pair search with interaction
 * masks (L131-L133, L187), exclusion masks (L135), list splitting/sorting (L199-L201).
 * Sets inner list := outer list.  NB_ERR_CUTOFF unless rc <= rlist_outer <= min(L)/2;
 * NB_ERR_BOX for a non-positive box; NB_ERR_ARG if an atom type is outside [0, ntypes).
 * All of it runs on the device; list buffers are sized from the previous search with head-room and
 * the stream is synchronised ONCE, at the end, to read the list sizes back (the first search of a
 * context, and a search whose list outgrew the buffers, synchronise stage by stage). */
int nb_search(nb_ctx*, float rlist_outer);

/* (a6) Dynamic pruning (L187-L193): recomputes the inner interaction mask of rolling part
 * `part` of `nparts` of the outer list from the current coordinates: a cluster pair stays
 * iff some atom pair is closer than rlist_inner.  Needs rc <= rlist_inner <= rlist_outer,
 * 0 <= part < nparts; nparts = 1 prunes everything. */
int nb_prune(nb_ctx*, float rlist_inner, int part, int nparts);
/* Same prune, scheduled "between force computations" so that it overlaps other work:
 * the kernel runs on a second stream of the library, concurrently with whatever the caller enqueues
 * next (the nb_forces of the same step), reads the coordinates of the last nb_put_atoms, and writes
 * the part into a second copy of the inner list.  The part switches to the new list at the NEXT
 * nb_put_atoms (which waits for the prune): the nb_forces calls before it still use the previous
 * list of that part, those after it the new one.  The list therefore serves one step longer than
 * with nb_prune: choose rlist_inner - rc for nparts + 1 steps of motion.  nparts <= 32. */
int nb_prune_overlapped(nb_ctx*, float rlist_inner, int part, int nparts);

/* (a7)-(a8) Forces over the inner list.  f [dev] natoms*3 fp32 in the caller's atom order,
 * overwritten.  energies [dev] double[2] = {E_lj, E_coul} (kJ/mol) or NULL for the force-only
 * kernel flavour (L139).  virial [dev] double[9] row-major, Xi = -1/2 sum_pairs d (x) F, or
 * NULL; a non-NULL virial requires non-NULL energies. */
int nb_forces(nb_ctx*, float* f, double* energies, double* virial);
/* Same with host pointers; synchronises before returning. */
int nb_forces_host(nb_ctx*, float* f, double* energies, double* virial);
/* First use of a freshly searched list ("Initial pruning is done the first time the
 * list is processed by a special version of the kernel (using warp collectives for low extra cost),
 * and the pruned list is reused for consecutive MD steps"): ONE kernel walks the OUTER list, computes
 * the forces (and energies / virial, as nb_forces) and writes the whole inner list for rlist_inner from
 * the distances it evaluates anyway.  Equivalent to nb_prune(rlist_inner, 0, 1) followed by nb_forces:
 * same inner list bit for bit, forces equal up to summation order.  Same argument rules as nb_prune / nb_forces. */
int nb_forces_prune(nb_ctx*, float rlist_inner, float* f, double* energies, double* virial);

/* Local / non-local split of the non-bonded work (with domain decomposition "interactions with particles
 * not local to the domain depend on halo exchange.  This is handled by splitting non-bonded work into two kernels: one for
 * local-only interactions and one for interactions that involve non-local particles. ... launch non-local work in a high
 * priority stream to preempt the local kernel and return remote forces early, while the local kernel execution can overlap
 * with communication").  This library is the kernel side of that design on ONE GPU; the halo exchange itself (which atoms
 * a rank receives, the transfers) is the caller's.
 *   nb_set_local(nlocal): atoms [0, nlocal) of the caller's order are the domain's LOCAL (home) atoms, atoms
 *     [nlocal, natoms) its NON-LOCAL (halo) atoms.  Takes effect at the next nb_search (required: the current list is
 *     dropped), which grids the two classes separately so that every cluster is purely local or non-local; lists, prune,
 *     nb_forces, nb_step work as before on the union.  nlocal = natoms (the default) switches the split off.
 *   nb_forces_nonlocal(f, energies, virial): enqueues, on the library's HIGH-PRIORITY stream (ordered after everything enqueued on the
 *     context's stream so far), the force kernel over the pairs of the inner list that involve at least one non-local
 *     atom, then writes the finished forces of the non-local atoms to f[nlocal .. natoms) ([dev] natoms*3 as in nb_forces;
 *     rows of local atoms are not touched by this call).  Every atom pair of the system is in exactly one of the two
 *     kernels (which non-local/non-local pairs a rank owns is a decomposition rule the caller applies by what it puts in).
 *   nb_sync_nonlocal(): blocks the host until those non-local forces are complete (the point where a caller sends them
 *     back to their home ranks while the local kernel still runs).
 *   nb_forces_local(f): enqueues the local-local kernel on the context's stream -- it runs next to the non-local one -- and,
 *     after both kernels, writes the forces of the local atoms (local-local + their share of the non-local pairs) to
 *     f[0 .. nlocal).  Must follow nb_forces_nonlocal (NB_ERR_STATE otherwise; so do nb_put_atoms, nb_search, nb_prune and
 *     nb_forces between the two calls: nothing may overtake the non-local kernel); after it f equals what nb_forces(f, NULL,
 *     NULL) gives, up to the order of the atomic adds.  energies / virial as in nb_forces ([dev]; NULL: the force-only
 *     kernel flavour): both kernels add into them, they are complete after nb_forces_local.  Not available while stage
 *     timing is on. */
int nb_set_local(nb_ctx*, int32_t nlocal);
int nb_forces_nonlocal(nb_ctx*, float* f, double* energies, double* virial);
int nb_forces_local(nb_ctx*, float* f);
int nb_sync_nonlocal(nb_ctx*);
/* Introspection of the split after nb_search: clusters [0, nclusters_local) hold local atoms only, the others non-local
 * atoms only; the force kernel's segment order (the order nb_inner_dump walks) has the nseg_local local-local segments
 * first, then the nseg - nseg_local segments that involve a non-local cluster. */
int nb_split_info(nb_ctx*, int32_t* nlocal, int32_t* nclusters_local, int32_t* nseg_local, int32_t* nseg);

/* nb_forces for callers that cannot call cudaMalloc (a stream under CUDA graph capture, a tight serving loop, a harness
 * that forbids it): same arguments, same kernels, same results up to the order of the atomic adds, but the call allocates
 * NOTHING -- no cudaMalloc / cudaFree, no event creation, no allocating library routine.  The force kernel's scratch (the
 * cluster-order force accumulator and the per-shift force sums of the virial: i and j forces are
 * accumulated on the device and reduced once) lives in one static device array of NB_STATIC_SCRATCH_BYTES inside the
 * library instead of the context's own buffers; every GPU that loads the library holds it until the process exits.
 * Limit: the bound on the system's atom slots, 64 * (natoms/64 + columns of the search grid), a few per cent above
 * natoms, must not exceed NB_STATIC_MAX_SLOTS -- about 245 000 atoms; beyond it the call returns NB_ERR_OVERFLOW with a
 * message and does nothing.  The array is shared by every context on the device and keeps the last call's contents: each
 * call clears what it uses on its stream first, and two calls that overlap on the GPU (two contexts on different streams)
 * RACE -- serialise them.  No stage timing is recorded for this call.  Its device address is resolved per device at
 * nb_init (cudaGetSymbolAddress); if that failed the call returns NB_ERR_CUDA.  Call-order rules as nb_forces. */
#define NB_STATIC_MAX_SLOTS 262144
#define NB_STATIC_SCRATCH_BYTES ((64 + NB_STATIC_MAX_SLOTS + 8 * 1024) * 16)   /* 4 326 400 B */
int nb_forces_static(nb_ctx*, float* f, double* energies, double* virial);

/* One inner step of the schedule as ONE call: nb_put_atoms(x, NULL, NULL, the box of the last search) +
 * nb_prune(rlist_inner, part, nparts) + nb_forces(f, NULL, NULL): the same kernels in the same order, so the same inner
 * list bit for bit and the same forces up to the order of the atomic adds.
 * From the second use of a (part, nparts, rlist_inner) on a given list the three stages are enqueued as one CUDA graph
 * launch (captured once, updated in place after every search; x and f are patched into it at each call), which is what
 * makes small systems, whose step is a handful of 3-30 us kernels, launch-bound no longer (the
 * strong-scaling regime of a few hundred atoms per SM).  x [dev] natoms*3 continuous coordinates, f [dev] natoms*3.
 * Needs a valid list and an unchanged box (NB_ERR_STATE otherwise); other errors as nb_prune / nb_forces.
 * With stage timing on, an overlapped prune in flight or more than 32 parts it simply runs the three calls. */
int nb_step(nb_ctx*, const float* x, float rlist_inner, int part, int nparts, float* f);

/* One inner step with HOST buffers (the positions-in / forces-out exchange of PAPER.md L105), with the rolling prune
 * hidden in the transfer gaps (L193: pruning "scheduled in chunks between force computations ... allows it to overlap
 * other work"): x [host] natoms*3 is copied in (the copy runs next to a prune still in flight from the previous call),
 * the forces over the current inner list are computed and copied to f [host] natoms*3, and the prune of `part` is
 * started on the library's second stream right after the force kernel -- it overlaps the device-to-host copy, whatever
 * the host does between two calls, and the next host-to-device copy.  Returns when f is complete (the prune may still
 * be running).  As with nb_prune_overlapped the part pruned here, on THIS call's coordinates, is first used by the next
 * call: pass the part the next step would have pruned, and choose rlist_inner - rc for nparts + 1 steps of motion. */
int nb_step_host(nb_ctx*, const float* x, float* f, float rlist_inner, int part, int nparts);

void nb_free(nb_ctx*);
const char* nb_last_error(const nb_ctx*);

/* ---- introspection: for parity tests and statistics only; these synchronise ---- */
int nb_get_layout(nb_ctx*, int32_t* cluster_size, int32_t* nclusters, int32_t* nsuper, int32_t* nslots);
/* atom_of_slot [dev] nslots (-1 = padding); xq [dev] nslots*4 (x,y,z,q as used by the kernels:
 * wrapped at the last search, then moved by nb_put_atoms).  Either may be NULL. */
int nb_get_slots(nb_ctx*, int32_t* atom_of_slot, float* xq);
/* Number of listed cluster pairs (ci,cj,shift): which = 0 outer, 1 inner. */
int nb_list_count(nb_ctx*, int which, int64_t* n);
/* Dumps the list in its stored order (deterministic).  All arrays [dev] with n entries (n from
 * nb_list_count); any may be NULL.  shift: 0..26 as defined by NB_SHIFT_CENTER, displacing the
 * i-cluster: d = x_a + s L - x_b.  pairmask bit a*8+b = 1: atoms a of ci and b of cj interact
 * (both real, not excluded, not the same atom, and b > a when ci == cj at zero shift).
 * part: rolling part of the entry under the nparts of the last nb_prune (0 before any prune). */
int nb_list_dump(nb_ctx*, int which, int32_t* ci, int32_t* cj, int32_t* shift, uint64_t* pairmask,
                 int32_t* part);
/* Dumps the COMPACT inner list the force kernel streams (for parity tests; slow, synchronises).
 * HOST arrays of *n entries, any may be NULL; call with all NULL to get *n.  Entry k: i-cluster ci[k],
 * shift[k] (as in nb_list_dump), kind[k] = 0: entry[k] is the SLOT of one j atom (of a cluster pair without a
 * mask: the list is kept at single-j-atom granularity, the atom is listed iff it is within rlist_inner of an atom of ci);
 * kind[k] = 1: entry[k] is a whole j-cluster cj whose pair with ci carries a mask; part[k]: rolling
 * part of the entry under the nparts of the last prune call.  Padding (dummy) entries are left out.
 * An overlapped prune still in flight is joined first. */
int nb_inner_dump(nb_ctx*, int64_t* n, int32_t* ci, int32_t* entry, int32_t* shift, int32_t* kind, int32_t* part);
int nb_get_stats(nb_ctx*, nb_stats* out);
/* Measures the device's FP32 FMA issue peak with a register-resident FFMA chain kernel
 * (MEASURED_PEAKS.json has no FP32 entry).  Returns lane-FMA/s in *fma_per_s. */
int nb_measure_fp32_peak(nb_ctx*, double* fma_per_s);
/* What the FP32 pipe really sustains for the instruction forms of the force kernel (the FP32x2 forms are bound by
 * register-file bandwidth, not by the 128 lanes): cycles per warp instruction per SM sub-partition, 4 warps per
 * sub-partition, everything in registers, at the device's nominal SM clock.  cycles[4] (host) = { scalar FFMA with three
 * different register operands, FFMA2 with three different register pairs, FFMA2 pair * pair + constant-bank operand,
 * FMUL2 with two different register pairs }.  bench.py reports them next to the roofline.  Synchronises. */
int nb_measure_fp32_pipe(nb_ctx*, double* cycles);
/* Counts, over the current inner list and coordinates, the atom pairs with r^2 < rc^2 that
 * interact (*n_interacting: the paper's "effective" pair count) and those
 * that are force-field exclusions (*n_excluded; they contribute only the Ewald/RF correction).
 * Host outputs; either may be NULL.  Synchronises. */
int nb_count_pairs(nb_ctx*, int64_t* n_interacting, int64_t* n_excluded);
/* Atom-pair slots the force kernel evaluates over the current inner list (the paper's "raw" pair
 * count, L167): 8 slots (the 8 i atoms) per listed j atom of the cluster pairs without a mask; cluster pairs that carry
 * an exclusion mask stay whole, 64 slots.  Host output.  Synchronises. */
int nb_count_slots(nb_ctx*, int64_t* slots);

/* Per-stage device timing with CUDA events on the context's stream ("CUDA events
 * on the caller's stream").  Stage ids index the arrays of nb_timing_read. */
enum { NB_T_PUT = 0,      /* (a1) nb_put_atoms: copies + cluster-order refresh */
       NB_T_GRID = 1,     /* (a2) gridding + cluster sort */
       NB_T_SEARCH = 2,   /* (a3)+(a5) pair search count/fill passes, unit table upload */
       NB_T_MASKS = 3,    /* (a4) exclusion masks, (a5) compact inner list set-up and its launch order (+ list statistics) */
       NB_T_PRUNE = 4,    /* (a6) prune kernel */
       NB_T_FORCE = 5,    /* (a7) force kernel alone, force-only flavour */
       NB_T_REDUCE = 6,   /* (a8) gather to caller order, virial/energy finalisation */
       NB_T_FORCE_ENERGY = 7,   /* (a7) force kernel alone, force + energy (+ virial) flavour */
       NB_T_NKINDS = 8 };
/* on != 0: record an event pair around every stage from now on.  Off by default. */
int nb_timing_enable(nb_ctx*, int on);
/* Restricts the timing to the stages whose bit (1u << NB_T_*) is set in stage_mask (default: all).
 * Every timed stage costs two event records per call, about 1.5 us of stream time each on a B200:
 * time one stage when the surrounding step is being timed as well. */
int nb_timing_stages(nb_ctx*, unsigned stage_mask);
/* Synchronises the stream, then returns the accumulated milliseconds and number of timed
 * intervals per stage (host arrays of NB_T_NKINDS; either may be NULL); reset != 0 zeroes
 * the accumulators afterwards. */
int nb_timing_read(nb_ctx*, double* ms, int64_t* count, int reset);

#ifdef __cplusplus
}
#endif
#endif /* NB_B200_H */
