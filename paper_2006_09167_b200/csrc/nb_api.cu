// nb_api.cu -- the C ABI of include/nb.h: argument checking, state machine, parameter
// preparation and memory ownership.  All arithmetic of the method lives in the kernels of
// nb_grid.cu / nb_list.cu / nb_prune.cu / nb_force.cu.  Links the CUDA runtime only.
#include "nb_internal.h"
#include "ewald_corr_coeffs.h"

#include <math.h>
#include <stdarg.h>

#include <new>

int nb_fail(nb_ctx* c, int code, const char* fmt, ...)
{
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

static bool finite_pos(float v) { return v > 0.f && isfinite(v); }

// Every entry point runs on the context's device whatever device is current in the calling thread,
// and leaves the caller's current device as it found it.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const nb_ctx* c)
    {
        if (!c) return;
        if (cudaGetDevice(&prev) == cudaSuccess && prev != c->prm.device) switched = cudaSetDevice(c->prm.device) == cudaSuccess;
    }
    ~DeviceGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
};

extern "C" int nb_init(const nb_params* p, nb_ctx** out)
{
    if (!p || !out) return NB_ERR_ARG;
    *out = nullptr;
    if (p->natoms <= 0 || p->ntypes <= 0 || p->ntypes > NB_MAX_TYPES || !p->lj_c6c12 || !finite_pos(p->rc)) return NB_ERR_ARG;
    if (p->coulomb != NB_COUL_EWALD && p->coulomb != NB_COUL_RF && p->coulomb != NB_COUL_NONE) return NB_ERR_ARG;
    if (p->excl_off && p->excl_off[p->natoms] > 0 && !p->excl_idx) return NB_ERR_ARG;
    int prev_device = -1;
    cudaGetDevice(&prev_device);
    if (cudaSetDevice(p->device) != cudaSuccess) return NB_ERR_CUDA;
    struct Restore { int d; ~Restore() { if (d >= 0) cudaSetDevice(d); } } restore{prev_device};
    nb_ctx* c = new (std::nothrow) nb_ctx();
    if (!c) return NB_ERR_NOMEM;
    c->err[0] = 0;
    memset(&c->st, 0, sizeof(c->st));
    c->prm = *p;
    c->prm.lj_c6c12 = nullptr; c->prm.excl_off = nullptr; c->prm.excl_idx = nullptr;
    c->stream = (cudaStream_t)p->stream;
    c->natoms = p->natoms;
    c->ntypes = p->ntypes;
    c->nlocal = p->natoms;         // no local / non-local split until nb_set_local
    nbi_static_scratch_setup(c);   // nb_forces_static: device address of the static scratch, once per device (never fails nb_init)
    if (cudaDeviceGetAttribute(&c->nsm, cudaDevAttrMultiProcessorCount, p->device) != cudaSuccess || c->nsm <= 0) c->nsm = 148;
    *out = c;   // returned even on failure below so that nb_last_error() can be read; nb_free() it

    // ---- interaction constants (fp64 on the host, stored fp32) ----
    const double rc = p->rc;
    const double epsfac = p->epsfac != 0.f ? (double)p->epsfac : 138.935458;   // reading A2
    double beta = 0.0;
    if (p->coulomb == NB_COUL_EWALD) {
        if (p->ewald_beta > 0.f) beta = p->ewald_beta;
        else {
            if (!(p->ewald_rtol > 0.f && p->ewald_rtol < 1.f)) return nb_fail(c, NB_ERR_ARG, "ewald_rtol must be in (0,1) when ewald_beta <= 0");
            double lo = 0.0, hi = 1.0;   // reading A3: erfc(beta*rc) = rtol
            while (erfc(hi * rc) > p->ewald_rtol) hi *= 2.0;
            for (int it = 0; it < 200; it++) {
                double mid = 0.5 * (lo + hi);
                if (erfc(mid * rc) > p->ewald_rtol) lo = mid; else hi = mid;
            }
            beta = 0.5 * (lo + hi);
        }
        if (beta * rc * beta * rc > (double)NB_EWALD_ZMAX)
            return nb_fail(c, NB_ERR_ARG, "(beta*rc)^2 = %g exceeds %g, the range of the Ewald correction fit", beta * rc * beta * rc, (double)NB_EWALD_ZMAX);
    }
    NbConst& K = c->kc;
    memset(&K, 0, sizeof(K));
    K.rc2 = p->rc * p->rc;
    if (p->rc_vdw < 0.f || p->rc_vdw > p->rc || !isfinite(p->rc_vdw))
        return nb_fail(c, NB_ERR_ARG, "rc_vdw = %g must be 0 (= rc) or in (0, rc = %g]", p->rc_vdw, p->rc);
    const double rcv = p->rc_vdw > 0.f ? (double)p->rc_vdw : rc;   // twin cut-offs: LJ below rc_vdw only
    c->twin = p->rc_vdw > 0.f && p->rc_vdw < p->rc;
    K.rcv2 = c->twin ? p->rc_vdw * p->rc_vdw : K.rc2;
    K.epsfac = (float)epsfac;
    K.beta = (float)beta; K.beta2 = (float)(beta * beta); K.beta3 = (float)(beta * beta * beta);
    K.ewald_shift = (p->coulomb == NB_COUL_EWALD && p->coul_modifier == NB_MOD_POTSHIFT) ? (float)(erfc(beta * rc) / rc) : 0.f;
    double krf = (p->eps_rf <= 0.f || isinf(p->eps_rf)) ? 1.0 / (2.0 * rc * rc * rc)
                                                         : ((double)p->eps_rf - 1.0) / ((2.0 * p->eps_rf + 1.0) * rc * rc * rc);   // reading A6
    K.krf = (float)krf; K.two_krf = (float)(2.0 * krf); K.crf = (float)(1.0 / rc + krf * rc * rc);
    K.lj_sh6 = p->lj_modifier == NB_MOD_POTSHIFT ? (float)pow(rcv, -6.0) : 0.f;
    K.lj_sh12 = p->lj_modifier == NB_MOD_POTSHIFT ? (float)pow(rcv, -12.0) : 0.f;
    K.ntypes1 = p->ntypes + 1;
    c->beta = (float)beta;
    c->beta_d = beta;
    c->st.ewald_beta = (float)beta;

    cudaStream_t st = c->stream;
    const int n = p->natoms, nt1 = p->ntypes + 1;
    std::vector<float2> tab((size_t)nt1 * nt1, make_float2(0.f, 0.f));
    for (int i = 0; i < p->ntypes; i++)
        for (int j = 0; j < p->ntypes; j++) {
            const float* e = p->lj_c6c12 + 2 * ((size_t)i * p->ntypes + j);
            tab[(size_t)i * nt1 + j] = make_float2(6.f * e[0], 12.f * e[1]);
        }
    NB_CUDA(c, c->ljtab.ensure(tab.size(), st));
    NB_CUDA(c, cudaMemcpyAsync(c->ljtab.p, tab.data(), tab.size() * sizeof(float2), cudaMemcpyHostToDevice, st));
    std::vector<int32_t> zero_off;
    const int32_t* eo = p->excl_off;
    if (!eo) { zero_off.assign(n + 1, 0); eo = zero_off.data(); }
    c->nexcl = eo[n];
    if (eo[0] != 0 || c->nexcl < 0) return nb_fail(c, NB_ERR_ARG, "excl_off must start at 0 and be non-decreasing");
    for (int i = 0; i < n; i++) {
        if (eo[i + 1] < eo[i]) return nb_fail(c, NB_ERR_ARG, "excl_off must be non-decreasing");
        for (int k = eo[i]; k < eo[i + 1]; k++)
            if (p->excl_idx[k] < 0 || p->excl_idx[k] >= n || p->excl_idx[k] == i)
                return nb_fail(c, NB_ERR_ARG, "exclusion %d of atom %d is out of range or a self entry", k, i);
    }
    // symmetric: the mask kernel walks each excluded pair from its lower index only
    for (int i = 0; i < n; i++)
        for (int k = eo[i]; k < eo[i + 1]; k++) {
            const int j = p->excl_idx[k];
            bool mirrored = false;
            for (int m = eo[j]; m < eo[j + 1] && !mirrored; m++) mirrored = p->excl_idx[m] == i;
            if (!mirrored) return nb_fail(c, NB_ERR_ARG, "exclusion (%d,%d) has no mirror entry (%d,%d)", i, j, j, i);
        }
    NB_CUDA(c, c->excl_off.ensure(n + 1, st));
    NB_CUDA(c, c->excl_idx.ensure(c->nexcl + 1, st));
    NB_CUDA(c, cudaMemcpyAsync(c->excl_off.p, eo, sizeof(int32_t) * (n + 1), cudaMemcpyHostToDevice, st));
    if (c->nexcl) NB_CUDA(c, cudaMemcpyAsync(c->excl_idx.p, p->excl_idx, sizeof(int32_t) * c->nexcl, cudaMemcpyHostToDevice, st));
    NB_CUDA(c, c->x.ensure((size_t)3 * n, st));
    NB_CUDA(c, c->q.ensure(n, st));
    NB_CUDA(c, c->type.ensure(n, st));
    NB_CUDA(c, cudaMalloc((void**)&c->tot_dev, sizeof(NbTotals)));
    NB_CUDA(c, cudaMallocHost((void**)&c->tot_host, sizeof(NbTotals)));
    memset(c->tot_host, 0, sizeof(NbTotals));
    NB_CUDA(c, cudaMemsetAsync(c->tot_dev, 0, sizeof(NbTotals), st));
    NB_CUDA(c, cudaStreamSynchronize(st));   // host staging vectors go out of scope
    return NB_OK;
}

static int put_atoms_common(nb_ctx* c, const float* x, const float* q, const int32_t* type, const float box[3], cudaMemcpyKind kind)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    if (!x || !box) return nb_fail(c, NB_ERR_ARG, "nb_put_atoms: null argument");
    if (c->nl_pending) return nb_fail(c, NB_ERR_STATE, "nb_put_atoms between nb_forces_nonlocal and nb_forces_local (the non-local kernel may still read the coordinates)");
    if ((!q || !type) && !c->have_atoms)
        return nb_fail(c, NB_ERR_ARG, "nb_put_atoms: q and type may be NULL only after a call that passed them");
    for (int k = 0; k < 3; k++)
        if (!finite_pos(box[k])) return nb_fail(c, NB_ERR_BOX, "box[%d] = %g is not positive", k, box[k]);
    cudaStream_t st = c->stream;
    const int n = c->natoms;
    NbStageTimer tm(c, NB_T_PUT);
    bool device = kind == cudaMemcpyDeviceToDevice;
    if (!device && !q && !type && c->pending_part < 0) {
        // Positions only, from PINNED host memory (cudaHostAlloc / cudaHostRegister, as torch's pin_memory gives): the put
        // kernel reads them in place over PCIe, coalesced, and writes both the caller-order copy and the cluster-ordered
        // array -- one kernel instead of a staging copy followed by a refresh kernel.
        cudaPointerAttributes pa;
        if (cudaPointerGetAttributes(&pa, x) == cudaSuccess && pa.type == cudaMemoryTypeHost && pa.devicePointer) {
            x = (const float*)pa.devicePointer;
            device = true;
        } else {
            cudaGetLastError();
        }
    }
    if (!device) {
        // (enqueued BEFORE the join below: the staging copy does not touch what an overlapped prune reads, so the
        // transfer and the prune run side by side)
        NB_CUDA(c, cudaMemcpyAsync(c->x.p, x, sizeof(float) * 3 * n, kind, st));
        if (q) NB_CUDA(c, cudaMemcpyAsync(c->q.p, q, sizeof(float) * n, kind, st));
        if (type) NB_CUDA(c, cudaMemcpyAsync(c->type.p, type, sizeof(int32_t) * n, kind, st));
    }
    // an overlapped prune reads the cluster-ordered coordinates this call overwrites: join it; its part flips to the new list here
    int rcp = nbi_commit_pending(c);
    if (rcp != NB_OK) return rcp;
    for (int k = 0; k < 3; k++) c->box[k] = box[k];
    c->have_atoms = true;
    c->atoms_since_search = true;
    bool refresh = false;
    if (c->have_grid) {
        if (box[0] != c->grid_box[0] || box[1] != c->grid_box[1] || box[2] != c->grid_box[2]) {
            c->have_list = false;   // a new box needs a new search
            c->have_grid = false;
        } else {
            refresh = true;
        }
    }
    if (device) return nbi_put_device(c, x, q, type, refresh);   // one launch: copies + refresh
    return refresh ? nbi_refresh_xq(c) : NB_OK;
}

extern "C" int nb_put_atoms(nb_ctx* c, const float* x, const float* q, const int32_t* type, const float box[3])
{
    return put_atoms_common(c, x, q, type, box, cudaMemcpyDeviceToDevice);
}

extern "C" int nb_put_atoms_host(nb_ctx* c, const float* x, const float* q, const int32_t* type, const float box[3])
{
    return put_atoms_common(c, x, q, type, box, cudaMemcpyHostToDevice);
}

static void step_graphs_refresh(nb_ctx* c);

extern "C" int nb_search(nb_ctx* c, float rlist_outer)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    if (!c->have_atoms) return nb_fail(c, NB_ERR_STATE, "nb_search before nb_put_atoms");
    if (c->nl_pending) return nb_fail(c, NB_ERR_STATE, "nb_search between nb_forces_nonlocal and nb_forces_local");
    const float minL = fminf(c->box[0], fminf(c->box[1], c->box[2]));
    if (!(rlist_outer >= c->prm.rc) || !(rlist_outer <= 0.5f * minL))
        return nb_fail(c, NB_ERR_CUTOFF, "rlist_outer = %g must satisfy rc = %g <= rlist_outer <= min(L)/2 = %g", rlist_outer, c->prm.rc, 0.5f * minL);
    c->have_list = false;
    int rc = nbi_search(c, rlist_outer);
    if (rc == NB_OK) step_graphs_refresh(c);   // the step graphs of the previous list, re-captured for this one
    return rc;
}

static int prune_checks(nb_ctx* c, float rlist_inner, int part, int nparts)
{
    if (!c->have_list) return nb_fail(c, NB_ERR_STATE, "nb_prune without a valid list (call nb_search)");
    if (c->nl_pending) return nb_fail(c, NB_ERR_STATE, "nb_prune between nb_forces_nonlocal and nb_forces_local (the non-local kernel may still read the list)");
    if (nparts < 1 || part < 0 || part >= nparts) return nb_fail(c, NB_ERR_ARG, "nb_prune: part %d of %d", part, nparts);
    if (!(rlist_inner >= c->prm.rc) || !(rlist_inner <= c->rlist_outer))
        return nb_fail(c, NB_ERR_CUTOFF, "rlist_inner = %g must satisfy rc = %g <= rlist_inner <= rlist_outer = %g", rlist_inner, c->prm.rc, c->rlist_outer);
    return NB_OK;
}

extern "C" int nb_prune(nb_ctx* c, float rlist_inner, int part, int nparts)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    int rc = prune_checks(c, rlist_inner, part, nparts);
    return rc != NB_OK ? rc : nbi_prune(c, rlist_inner, part, nparts);
}

extern "C" int nb_prune_overlapped(nb_ctx* c, float rlist_inner, int part, int nparts)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    int rc = prune_checks(c, rlist_inner, part, nparts);
    return rc != NB_OK ? rc : nbi_prune_overlapped(c, rlist_inner, part, nparts);
}

extern "C" int nb_forces(nb_ctx* c, float* f, double* energies, double* virial)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    if (!f) return nb_fail(c, NB_ERR_ARG, "nb_forces: f is null");
    if (virial && !energies) return nb_fail(c, NB_ERR_ARG, "nb_forces: virial needs energies (same kernel flavour)");
    if (!c->have_list) return nb_fail(c, NB_ERR_STATE, "nb_forces without a valid list (call nb_search)");
    if (c->nl_pending) return nb_fail(c, NB_ERR_STATE, "nb_forces between nb_forces_nonlocal and nb_forces_local");
    return nbi_forces(c, f, energies, virial);
}

// ---- local / non-local split ----
extern "C" int nb_set_local(nb_ctx* c, int32_t nlocal)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    if (nlocal < 1 || nlocal > c->natoms) return nb_fail(c, NB_ERR_ARG, "nb_set_local: nlocal = %d outside [1, %d]", nlocal, c->natoms);
    if (c->nl_pending) return nb_fail(c, NB_ERR_STATE, "nb_set_local between nb_forces_nonlocal and nb_forces_local");
    int rc = nbi_commit_pending(c);
    if (rc != NB_OK) return rc;
    if (nlocal != c->nlocal) {
        c->nlocal = nlocal;
        c->have_list = false;   // the grid changes: a new search is needed
        c->have_grid = false;
        c->cold = true;         // and its buffers are sized afresh
    }
    return nlocal < c->natoms ? nbi_split_setup(c) : NB_OK;
}

extern "C" int nb_forces_nonlocal(nb_ctx* c, float* f, double* energies, double* virial)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    if (!f) return nb_fail(c, NB_ERR_ARG, "nb_forces_nonlocal: f is null");
    if (virial && !energies) return nb_fail(c, NB_ERR_ARG, "nb_forces_nonlocal: virial needs energies (same kernel flavour)");
    if (!c->have_list) return nb_fail(c, NB_ERR_STATE, "nb_forces_nonlocal without a valid list (call nb_search)");
    if (c->nl_pending) return nb_fail(c, NB_ERR_STATE, "nb_forces_nonlocal twice without nb_forces_local");
    if (c->timing) return nb_fail(c, NB_ERR_STATE, "nb_forces_nonlocal: stage timing is not available for the split kernels");
    int rc = nbi_commit_pending(c);
    return rc != NB_OK ? rc : nbi_forces_nonlocal(c, f, energies, virial);
}

extern "C" int nb_forces_local(nb_ctx* c, float* f)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    if (!f) return nb_fail(c, NB_ERR_ARG, "nb_forces_local: f is null");
    if (!c->nl_pending) return nb_fail(c, NB_ERR_STATE, "nb_forces_local without a preceding nb_forces_nonlocal");
    return nbi_forces_local(c, f);
}

extern "C" int nb_sync_nonlocal(nb_ctx* c)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    return nbi_sync_nonlocal(c);
}

extern "C" int nb_split_info(nb_ctx* c, int32_t* nlocal, int32_t* nclusters_local, int32_t* nseg_local, int32_t* nseg)
{
    if (!c) return NB_ERR_ARG;
    if (!c->have_list) return nb_fail(c, NB_ERR_STATE, "nb_split_info without a valid list (call nb_search)");
    if (nlocal) *nlocal = c->nlocal;
    if (nclusters_local) *nclusters_local = c->nsc_local * NB_SUPER_SIZE;
    if (nseg_local) *nseg_local = c->nseg_local;
    if (nseg) *nseg = c->nseg_launch;
    return NB_OK;
}

extern "C" int nb_forces_static(nb_ctx* c, float* f, double* energies, double* virial)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    if (!f) return nb_fail(c, NB_ERR_ARG, "nb_forces_static: f is null");
    if (virial && !energies) return nb_fail(c, NB_ERR_ARG, "nb_forces_static: virial needs energies (same kernel flavour)");
    if (!c->have_list) return nb_fail(c, NB_ERR_STATE, "nb_forces_static without a valid list (call nb_search)");
    if (c->nl_pending) return nb_fail(c, NB_ERR_STATE, "nb_forces_static between nb_forces_nonlocal and nb_forces_local");
    return nbi_forces_static(c, f, energies, virial);
}

extern "C" int nb_forces_prune(nb_ctx* c, float rlist_inner, float* f, double* energies, double* virial)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    if (!f) return nb_fail(c, NB_ERR_ARG, "nb_forces_prune: f is null");
    if (virial && !energies) return nb_fail(c, NB_ERR_ARG, "nb_forces_prune: virial needs energies (same kernel flavour)");
    int rc = prune_checks(c, rlist_inner, 0, 1);
    if (rc != NB_OK) return rc;
    if ((rc = nbi_commit_pending(c)) != NB_OK) return rc;
    return nbi_forces(c, f, energies, virial, rlist_inner);
}

// ---- nb_step -------------------------------------------------------------------------------------------
static int step_plain(nb_ctx* c, const float* x, float rlist_inner, int part, int nparts, float* f)
{
    int rc = nbi_commit_pending(c);
    if (rc != NB_OK) return rc;
    c->atoms_since_search = true;
    if ((rc = nbi_put_device(c, x, nullptr, nullptr, true)) != NB_OK) return rc;
    if ((rc = nbi_prune(c, rlist_inner, part, nparts)) != NB_OK) return rc;
    return nbi_forces(c, f, nullptr, nullptr);
}

static void step_graph_release(nb_ctx::StepGraph& g)
{
    if (g.exec) cudaGraphExecDestroy(g.exec);
    if (g.graph) cudaGraphDestroy(g.graph);
    g.exec = nullptr;
    g.graph = nullptr;
    g.put = g.gather = nullptr;
}

// Captures put + prune + forces for this key on the private stream and instantiates (or updates) the executable graph.
static int step_capture(nb_ctx* c, nb_ctx::StepGraph& g, const float* x, float* f)
{
    if (!c->capture_stream && cudaStreamCreateWithFlags(&c->capture_stream, cudaStreamNonBlocking) != cudaSuccess) return NB_ERR_CUDA;
    const nb_stats saved = c->st;
    cudaStream_t user = c->stream;
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(c->capture_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) return NB_ERR_CUDA;
    c->stream = c->capture_stream;
    int rc = step_plain(c, x, g.rl, g.part, g.nparts, f);
    c->stream = user;
    const cudaError_t ee = cudaStreamEndCapture(c->capture_stream, &graph);
    c->st = saved;   // nothing ran: the counters move when the graph is launched
    if (rc != NB_OK || ee != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        return NB_ERR_CUDA;
    }
    cudaGraphNode_t nodes[16];
    size_t nn = 16;
    cudaGraphNode_t put = nullptr, gather = nullptr;
    if (cudaGraphGetNodes(graph, nodes, &nn) != cudaSuccess) { cudaGraphDestroy(graph); return NB_ERR_CUDA; }
    for (size_t i = 0; i < nn && i < 16; i++) {
        cudaGraphNodeType ty;
        cudaKernelNodeParams kp;
        if (cudaGraphNodeGetType(nodes[i], &ty) != cudaSuccess || ty != cudaGraphNodeTypeKernel) continue;
        if (cudaGraphKernelNodeGetParams(nodes[i], &kp) != cudaSuccess) continue;
        if (kp.func == nbi_put_kernel()) put = nodes[i];
        if (kp.func == nbi_gather4_kernel()) gather = nodes[i];
    }
    if (!put || !gather) { cudaGraphDestroy(graph); return NB_ERR_CUDA; }
    if (g.exec) {
        // Same topology as before the search: update the executable graph in place.  Node handles used with an executable
        // graph must be those of the graph it was instantiated from, so that graph stays, and its put / gather nodes take
        // over the new parameter blocks (they are what nb_step patches x and f into).
        cudaGraphExecUpdateResultInfo info;
        cudaKernelNodeParams kput, kgat;
        if (cudaGraphExecUpdate(g.exec, graph, &info) == cudaSuccess && cudaGraphKernelNodeGetParams(put, &kput) == cudaSuccess &&
            cudaGraphKernelNodeGetParams(gather, &kgat) == cudaSuccess && cudaGraphKernelNodeSetParams(g.put, &kput) == cudaSuccess &&
            cudaGraphKernelNodeSetParams(g.gather, &kgat) == cudaSuccess) {
            cudaGraphDestroy(graph);
            return NB_OK;
        }
        cudaGetLastError();
        step_graph_release(g);
    }
    if (cudaGraphInstantiate(&g.exec, graph, 0) != cudaSuccess) {
        cudaGetLastError();
        cudaGraphDestroy(graph);
        g.exec = nullptr;
        return NB_ERR_CUDA;
    }
    g.graph = graph;   // kept: node handles and the parameter blocks patched at every launch live in it
    g.put = put;
    g.gather = gather;
    return NB_OK;
}

// After a search: the graphs that were in use on the previous list are brought up to date here, once per list
// lifetime, instead of on their next use (a capture is ~50 us of host time that a step should not wait for).
static void step_graphs_refresh(nb_ctx* c)
{
    if (c->timing) return;
    const int64_t gen = c->st.search_count;
    for (auto& g : c->step_graphs) {
        if (!g.exec || g.broken || g.rl > c->rlist_outer || g.rl < c->prm.rc) continue;
        if (nbi_prepare_parts(c, g.nparts) != NB_OK) { g.broken = true; continue; }   // part tables and launch orders of this list
        if (step_capture(c, g, c->x.p, c->x.p) != NB_OK) { g.broken = true; continue; }   // (x and f are patched at every launch)
        g.warm_search = g.graph_search = gen;
    }
}

extern "C" int nb_step(nb_ctx* c, const float* x, float rlist_inner, int part, int nparts, float* f)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    if (!x || !f) return nb_fail(c, NB_ERR_ARG, "nb_step: null argument");
    if (!c->have_list || !c->have_grid) return nb_fail(c, NB_ERR_STATE, "nb_step without a valid list (call nb_search)");
    if (c->box[0] != c->grid_box[0] || c->box[1] != c->grid_box[1] || c->box[2] != c->grid_box[2])
        return nb_fail(c, NB_ERR_STATE, "nb_step: the box changed since the search (nb_put_atoms + nb_search first)");
    int rc = prune_checks(c, rlist_inner, part, nparts);
    if (rc != NB_OK) return rc;
    // the graph covers the steady state only: no stage timing, no overlapped prune in flight, at most 32 parts
    if (c->timing || nparts > 32 || c->pending_part >= 0 || c->bufmask) return step_plain(c, x, rlist_inner, part, nparts, f);
    nb_ctx::StepGraph* g = nullptr;
    for (auto& e : c->step_graphs)
        if (e.part == part && e.nparts == nparts && e.rl == rlist_inner) g = &e;
    if (!g) {
        g = &c->step_graphs[c->step_graph_next];
        c->step_graph_next = (c->step_graph_next + 1) % 8;
        step_graph_release(*g);
        *g = nb_ctx::StepGraph();
        g->part = part; g->nparts = nparts; g->rl = rlist_inner;
    }
    const int64_t gen = c->st.search_count;
    if (g->broken || g->warm_search != gen) {   // first use of this key on this list: the plain path sets everything up
        g->warm_search = gen;
        return step_plain(c, x, rlist_inner, part, nparts, f);
    }
    if (g->graph_search != gen) {
        if (step_capture(c, *g, x, f) != NB_OK) {
            g->broken = true;
            return step_plain(c, x, rlist_inner, part, nparts, f);
        }
        g->graph_search = gen;
    }
    // patch the caller's pointers into the put (argument 1: x) and gather (argument 3: f) nodes
    cudaKernelNodeParams kp;
    void* args[16];
    NB_CUDA(c, cudaGraphKernelNodeGetParams(g->put, &kp));
    for (int i = 0; i < 11; i++) args[i] = kp.kernelParams[i];
    args[1] = (void*)&x;
    kp.kernelParams = args;
    NB_CUDA(c, cudaGraphExecKernelNodeSetParams(g->exec, g->put, &kp));
    NB_CUDA(c, cudaGraphKernelNodeGetParams(g->gather, &kp));
    for (int i = 0; i < 4; i++) args[i] = kp.kernelParams[i];
    args[3] = (void*)&f;
    kp.kernelParams = args;
    NB_CUDA(c, cudaGraphExecKernelNodeSetParams(g->exec, g->gather, &kp));
    NB_CUDA(c, cudaGraphLaunch(g->exec, c->stream));
    // what the three calls would have recorded on the host
    c->atoms_since_search = true;
    c->last_nparts = nparts;
    c->planes_dirty = true;
    c->st.prune_count++;
    c->st.force_count++;
    c->st.kernel_launches += 4;
    return NB_OK;
}

extern "C" int nb_step_host(nb_ctx* c, const float* x, float* f, float rlist_inner, int part, int nparts)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    if (!x || !f) return nb_fail(c, NB_ERR_ARG, "nb_step_host: null argument");
    if (!c->have_list || !c->have_grid) return nb_fail(c, NB_ERR_STATE, "nb_step_host without a valid list (call nb_search)");
    if (nparts > 32) return nb_fail(c, NB_ERR_ARG, "nb_step_host: at most 32 rolling parts (got %d)", nparts);
    int rc = prune_checks(c, rlist_inner, part, nparts);
    if (rc != NB_OK) return rc;
    const float box[3] = {c->box[0], c->box[1], c->box[2]};
    if ((rc = put_atoms_common(c, x, nullptr, nullptr, box, cudaMemcpyHostToDevice)) != NB_OK) return rc;   // joins the previous prune
    if (!c->have_list) return nb_fail(c, NB_ERR_STATE, "nb_step_host: the box changed since the search");
    cudaStream_t st = c->stream;
    NB_CUDA(c, c->stage_f.ensure((size_t)3 * c->natoms, st));
    if ((rc = nbi_forces(c, c->stage_f.p, nullptr, nullptr)) != NB_OK) return rc;
    if ((rc = nbi_prune_overlapped(c, rlist_inner, part, nparts)) != NB_OK) return rc;   // forks here: after the force kernel and the gather
    NB_CUDA(c, cudaMemcpyAsync(f, c->stage_f.p, sizeof(float) * 3 * c->natoms, cudaMemcpyDeviceToHost, st));
    NB_CUDA(c, cudaStreamSynchronize(st));   // the forces are on the host; the prune may still be running
    return NB_OK;
}

extern "C" int nb_forces_host(nb_ctx* c, float* f, double* energies, double* virial)
{
    if (!c) return NB_ERR_ARG;
    DeviceGuard guard(c);
    if (!f) return nb_fail(c, NB_ERR_ARG, "nb_forces_host: f is null");
    cudaStream_t st = c->stream;
    NB_CUDA(c, c->stage_f.ensure((size_t)3 * c->natoms, st));
    NB_CUDA(c, c->stage_ev.ensure(16, st));
    int rc = nb_forces(c, c->stage_f.p, energies ? c->stage_ev.p : nullptr, virial ? c->stage_ev.p + 2 : nullptr);
    if (rc != NB_OK) return rc;
    NB_CUDA(c, cudaMemcpyAsync(f, c->stage_f.p, sizeof(float) * 3 * c->natoms, cudaMemcpyDeviceToHost, st));
    if (energies) NB_CUDA(c, cudaMemcpyAsync(energies, c->stage_ev.p, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (virial) NB_CUDA(c, cudaMemcpyAsync(virial, c->stage_ev.p + 2, 9 * sizeof(double), cudaMemcpyDeviceToHost, st));
    NB_CUDA(c, cudaStreamSynchronize(st));
    return NB_OK;
}

extern "C" void nb_free(nb_ctx* c)
{
    if (!c) return;
    DeviceGuard guard(c);
    if (c->side_stream) cudaStreamSynchronize(c->side_stream);
    cudaStreamSynchronize(c->stream);
    if (c->stream_hp) cudaStreamSynchronize(c->stream_hp);
    nbi_split_free(c);
    if (c->side_stream) cudaStreamDestroy(c->side_stream);
    for (auto& g : c->step_graphs) step_graph_release(g);
    if (c->capture_stream) cudaStreamDestroy(c->capture_stream);
    if (c->ev_main) cudaEventDestroy(c->ev_main);
    if (c->ev_side) cudaEventDestroy(c->ev_side);
    if (c->tot_dev) cudaFree(c->tot_dev);
    if (c->tot_host) cudaFreeHost(c->tot_host);
    for (auto& r : c->tim_open) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
    for (auto e : c->tim_pool) cudaEventDestroy(e);
    c->x.release(); c->q.release(); c->type.release();
    c->stage_x.release(); c->stage_q.release(); c->stage_f.release(); c->stage_type.release(); c->stage_ev.release();
    c->excl_off.release(); c->excl_idx.release(); c->ljtab.release();
    c->col_count.release(); c->col_atom_off.release(); c->col_sc_off.release(); c->atom_col.release();
    c->atom_rank.release(); c->col_atoms.release(); c->image.release(); c->xw_atom.release();
    c->xq.release(); c->type_slot.release(); c->atom_of_slot.release(); c->slot_of_atom.release();
    c->bb_lo.release(); c->bb_hi.release(); c->sbb_lo.release(); c->sbb_hi.release(); c->f4.release();
    c->ent_count.release(); c->ent_jbegin.release(); c->jl.release(); c->imask_outer.release();
    c->plane_outer.release(); c->plane_inner.release(); c->plane_excl.release(); c->batch_ent.release(); c->scan_tmp.release();
    c->scan_blk.release(); c->excl_masks.release(); c->counters.release(); c->units_canon.release();
    c->fshift.release(); c->unit_nsplit.release(); c->unit_off.release(); c->sort_hist.release(); c->seg_len.release();
    for (auto& po : c->prune_orders) po.d.release();
    c->il_off.release(); c->ilm_off.release(); c->seg_of_s0.release(); c->segd.release(); c->ol_cnt.release();
    c->olu.release(); c->olm.release(); c->ljrow.release(); c->seg_part.release();
    for (int b = 0; b < 2; b++) { c->seg_cnt[b].release(); c->il[b].release(); c->ilm[b].release(); }
    delete c;
}

extern "C" const char* nb_last_error(const nb_ctx* c) { return c ? c->err : "null context"; }

extern "C" int nb_get_layout(nb_ctx* c, int32_t* cluster_size, int32_t* nclusters, int32_t* nsuper, int32_t* nslots)
{
    DeviceGuard guard(c);
    if (!c) return NB_ERR_ARG;
    if (!c->have_grid) return nb_fail(c, NB_ERR_STATE, "no grid yet (call nb_search)");
    if (cluster_size) *cluster_size = NB_C;
    if (nclusters) *nclusters = c->nclusters;
    if (nsuper) *nsuper = c->nsc;
    if (nslots) *nslots = c->nslots;
    return NB_OK;
}

extern "C" int nb_get_slots(nb_ctx* c, int32_t* atom_of_slot, float* xq)
{
    DeviceGuard guard(c);
    if (!c) return NB_ERR_ARG;
    if (!c->have_grid) return nb_fail(c, NB_ERR_STATE, "no grid yet (call nb_search)");
    if (atom_of_slot) NB_CUDA(c, cudaMemcpyAsync(atom_of_slot, c->atom_of_slot.p, sizeof(int32_t) * c->nslots, cudaMemcpyDeviceToDevice, c->stream));
    if (xq) NB_CUDA(c, cudaMemcpyAsync(xq, c->xq.p, sizeof(float4) * c->nslots, cudaMemcpyDeviceToDevice, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    return NB_OK;
}

extern "C" int nb_list_count(nb_ctx* c, int which, int64_t* n)
{
    DeviceGuard guard(c);
    if (!c || !n) return NB_ERR_ARG;
    if (which != 0 && which != 1) return nb_fail(c, NB_ERR_ARG, "which must be 0 (outer) or 1 (inner)");
    if (!c->have_list) return nb_fail(c, NB_ERR_STATE, "no list yet (call nb_search)");
    return nbi_list_count(c, which, n);
}

extern "C" int nb_list_dump(nb_ctx* c, int which, int32_t* ci, int32_t* cj, int32_t* shift, uint64_t* pairmask, int32_t* part)
{
    DeviceGuard guard(c);
    if (!c) return NB_ERR_ARG;
    if (which != 0 && which != 1) return nb_fail(c, NB_ERR_ARG, "which must be 0 (outer) or 1 (inner)");
    if (!c->have_list) return nb_fail(c, NB_ERR_STATE, "no list yet (call nb_search)");
    return nbi_list_dump(c, which, ci, cj, shift, pairmask, part);
}

extern "C" int nb_get_stats(nb_ctx* c, nb_stats* out)
{
    DeviceGuard guard(c);
    if (!c || !out) return NB_ERR_ARG;
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    if (c->have_list) {
        int64_t n = 0;
        int rc = nbi_list_stats(c);
        if (rc != NB_OK) return rc;
        if ((rc = nbi_list_count(c, 1, &n)) != NB_OK) return rc;
        c->st.n_pairs_inner = n;
        int64_t slots = 0;
        if ((rc = nbi_count_slots(c, &slots)) != NB_OK) return rc;
        c->st.slots_last_forces = c->st.force_count ? slots : 0;
    }
    *out = c->st;
    return NB_OK;
}

extern "C" int nb_measure_fp32_peak(nb_ctx* c, double* fma_per_s)
{
    DeviceGuard guard(c);
    if (!c || !fma_per_s) return NB_ERR_ARG;
    return nbi_measure_fp32_peak(c, fma_per_s);
}

extern "C" int nb_measure_fp32_pipe(nb_ctx* c, double* cycles)
{
    DeviceGuard guard(c);
    if (!c || !cycles) return NB_ERR_ARG;
    return nbi_measure_fp32_pipe(c, cycles);
}

extern "C" int nb_count_pairs(nb_ctx* c, int64_t* n_interacting, int64_t* n_excluded)
{
    DeviceGuard guard(c);
    if (!c) return NB_ERR_ARG;
    if (!c->have_list) return nb_fail(c, NB_ERR_STATE, "no list yet (call nb_search)");
    return nbi_count_pairs(c, n_interacting, n_excluded);
}

extern "C" int nb_count_slots(nb_ctx* c, int64_t* slots)
{
    DeviceGuard guard(c);
    if (!c || !slots) return NB_ERR_ARG;
    if (!c->have_list) return nb_fail(c, NB_ERR_STATE, "no list yet (call nb_search)");
    return nbi_count_slots(c, slots);
}

extern "C" int nb_inner_dump(nb_ctx* c, int64_t* n, int32_t* ci, int32_t* entry, int32_t* shift, int32_t* kind, int32_t* part)
{
    DeviceGuard guard(c);
    if (!c || !n) return NB_ERR_ARG;
    if (!c->have_list) return nb_fail(c, NB_ERR_STATE, "no list yet (call nb_search)");
    return nbi_inner_dump(c, n, ci, entry, shift, kind, part);
}

extern "C" int nb_timing_enable(nb_ctx* c, int on)
{
    if (!c) return NB_ERR_ARG;
    c->timing = on != 0;
    return NB_OK;
}

extern "C" int nb_timing_stages(nb_ctx* c, unsigned stage_mask)
{
    if (!c) return NB_ERR_ARG;
    c->timing_mask = stage_mask;
    return NB_OK;
}

extern "C" int nb_timing_read(nb_ctx* c, double* ms, int64_t* count, int reset)
{
    DeviceGuard guard(c);
    if (!c) return NB_ERR_ARG;
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    for (auto& r : c->tim_open) {
        float t = 0.f;
        NB_CUDA(c, cudaEventElapsedTime(&t, r.e0, r.e1));
        c->tim_ms[r.kind] += t;
        c->tim_n[r.kind]++;
        c->tim_pool.push_back(r.e0);
        c->tim_pool.push_back(r.e1);
    }
    c->tim_open.clear();
    for (int k = 0; k < NB_T_NKINDS; k++) {
        if (ms) ms[k] = c->tim_ms[k];
        if (count) count[k] = c->tim_n[k];
        if (reset) { c->tim_ms[k] = 0.0; c->tim_n[k] = 0; }
    }
    return NB_OK;
}
