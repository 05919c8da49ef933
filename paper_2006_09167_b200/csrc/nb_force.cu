// nb_force.cu -- (a7) the cluster-pair force kernel and (a8) force reduction / outputs.
//
// interactions between i-clusters and a joint list of j-clusters, skipped
// per cluster pair through the interaction mask; Newton's third law so both i and j forces are
// reduced (L133); exclusions as bitmasks applied together with the cut-off (L135); analytical
// Ewald correction on FMA hardware (L137); one kernel per combination of electrostatics and
// energy/no-energy to avoid conditionals (L139).
//
// Thread mapping (differs from the paper's 8x4-per-warp tiles): a block is the
// 8 i-clusters of one super-cluster working through one chunk of the joint j list; warp w owns
// i-cluster w, whose 8 atoms sit in registers of every lane.  Lanes own j atoms: a step takes
// the next 4 j-clusters whose mask bit w is set (32 j atoms) and every lane evaluates its j
// atom against the 8 i atoms.  Consequences: no shuffle in the inner loop (the j force is
// private to its lane and leaves with ONE vector atomic per j atom per cluster pair, i.e.
// atomics at cluster granularity), no per-pair shared-memory load of i data, mask skipping
// costs nothing (set bits are compacted, not tested one by one), and the i forces (8 x 3
// registers) are reduced across lanes once per work unit.
#include "nb_internal.h"

#include "ewald_corr_coeffs.h"

namespace {

struct ForceArgs {
    const int4* units;
    const int2* jl;
    const uint32_t* plane;
    const uint32_t* plane_excl;
    const float4* xq;
    const int* type_slot;
    const float2* ljtab;
    const unsigned long long* masks;
    float4* f4;
    double* fshift;     // [27*3]
    double* energies;   // [2]
    NbConst kc;
};

__device__ __forceinline__ void red_add_v4(float4* addr, float x, float y, float z)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(x), "f"(y), "f"(z), "f"(0.0f)
                 : "memory");
}

// Single-instruction MUFU forms: the arguments are clamped away from zero/denormals by the
// caller (r^2 >= 1e-6, Q(z) >= 1), so the denormal fix-up code of rsqrtf()/__fdividef() is dead weight.
__device__ __forceinline__ float rsqrt_fast(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_fast(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// beta^3 h(z), h = P5/Q5 (ewald_corr_coeffs.h); z = beta^2 r^2; ewp[k] = beta^3 P_k.
__device__ __forceinline__ float ewald_bh(float z, const float (&ewp)[6])
{
    float p = ewp[5];
    p = fmaf(p, z, ewp[4]);
    p = fmaf(p, z, ewp[3]);
    p = fmaf(p, z, ewp[2]);
    p = fmaf(p, z, ewp[1]);
    p = fmaf(p, z, ewp[0]);
    float q = NB_EWC_Q5;
    q = fmaf(q, z, NB_EWC_Q4);
    q = fmaf(q, z, NB_EWC_Q3);
    q = fmaf(q, z, NB_EWC_Q2);
    q = fmaf(q, z, NB_EWC_Q1);
    q = fmaf(q, z, NB_EWC_Q0);
    return p * rcp_fast(q);
}

struct IAtoms {
    float x[8], y[8], z[8], q[8];
    int t[8];   // byte offset of the i atom's row in the shared LJ table
};

// One step: this lane's j atom (xj, byte offset tjb of its LJ column) against the 8 i atoms.
// MASKED: cbyte/mbyte carry the lane's 8 "counted"/"interacts" bits (reading A4: an excluded pair
// keeps the Ewald/RF correction, loses LJ and the 1/r part).
template <int COUL, bool ENERGY, bool MASKED>
__device__ __forceinline__ void pair_step(const NbConst& K, const char* __restrict__ s_ljb, const IAtoms& I,
                                          float (&fi)[24], float& elj, float& ecoul, const float4 xj, const int tjb,
                                          unsigned cbyte, unsigned mbyte, float& fjx, float& fjy, float& fjz)
{
    fjx = 0.f; fjy = 0.f; fjz = 0.f;
#pragma unroll
    for (int a = 0; a < 8; a++) {
        const float dx = I.x[a] - xj.x, dy = I.y[a] - xj.y, dz = I.z[a] - xj.z;
        float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        bool within = r2 < K.rc2;                            // A7: strict
        if (MASKED) within = within && ((cbyte >> a) & 1u);
        r2 = fmaxf(r2, 1e-6f);                               // keeps masked / padding pairs finite
        const float rinv = rsqrt_fast(r2);
        const float rinv2 = rinv * rinv;
        const float2 c = *reinterpret_cast<const float2*>(s_ljb + (I.t[a] + tjb));   // (6 c6, 12 c12)
        const float rinv6 = rinv2 * rinv2 * rinv2;
        const float flj = (c.y * rinv6 - c.x) * rinv6;
        const float qq = I.q[a] * xj.w;                      // epsfac folded into the i charge
        float t1 = fmaf(qq, rinv, flj);                      // (F_lj + A/r) r
        float mf = 1.f;
        if (MASKED) {
            mf = ((mbyte >> a) & 1u) ? 1.f : 0.f;            // excluded pair: only the correction term
            t1 *= mf;
        }
        float fs, bh = 0.f;
        if (COUL == NB_COUL_EWALD) {
            bh = ewald_bh(K.beta2 * r2, K.ewp);
            fs = fmaf(rinv2, t1, -qq * bh);                  // F/r = (F_lj r + A m/r)/r^2 - A beta^3 h
        } else {
            fs = fmaf(rinv2, t1, -qq * K.two_krf);           // F/r = ... - 2 A k_rf
        }
        fs = within ? fs : 0.f;
        fi[3 * a + 0] = fmaf(fs, dx, fi[3 * a + 0]);
        fi[3 * a + 1] = fmaf(fs, dy, fi[3 * a + 1]);
        fi[3 * a + 2] = fmaf(fs, dz, fi[3 * a + 2]);
        fjx = fmaf(-fs, dx, fjx);
        fjy = fmaf(-fs, dy, fjy);
        fjz = fmaf(-fs, dz, fjz);
        if (ENERGY) {
            const float vlj = c.y * (1.f / 12.f) * (rinv6 * rinv6 - K.lj_sh12) - c.x * (1.f / 6.f) * (rinv6 - K.lj_sh6);
            float vc;
            if (COUL == NB_COUL_EWALD) {
                // beta e(z) = r^2 beta^3 h(z) + beta (2/sqrt(pi)) exp(-z)
                const float be = fmaf(r2, bh, K.beta * 1.1283791671f * __expf(-K.beta2 * r2));
                vc = qq * (mf * (rinv - K.ewald_shift) - be);
            } else {
                vc = qq * (mf * rinv + K.krf * r2 - K.crf);
            }
            elj += within ? mf * vlj : 0.f;
            ecoul += within ? vc : 0.f;
        }
    }
}

template <int COUL, bool ENERGY>
__global__ void __launch_bounds__(256, 2) k_force(ForceArgs A)
{
    extern __shared__ float2 s_lj[];
    __shared__ int2 s_q[8][40];   // per-warp queue of cluster pairs without a mask for this i-cluster
    __shared__ int2 s_m[8][40];   // per-warp queue of cluster pairs with a non-trivial mask (and the unit's tail)
    const NbConst& K = A.kc;
    const char* s_ljb = reinterpret_cast<const char*>(s_lj);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 3, k = lane & 7;
    for (int i = threadIdx.x; i < K.ntypes1 * K.ntypes1; i += blockDim.x) s_lj[i] = A.ljtab[i];
    const int4 u = A.units[blockIdx.x];
    const int sci = u.w, h = u.x - sci * NB_NHALF, ci = sci * 8 + warp;
    const int sid = nb_half_shift_id(h);
    int sx, sy, sz;
    nb_shift_vec(sid, sx, sy, sz);
    IAtoms I;
#pragma unroll
    for (int a = 0; a < 8; a++) {
        const float4 v = A.xq[ci * 8 + a];
        I.x[a] = fmaf((float)sx, K.box[0], v.x);
        I.y[a] = fmaf((float)sy, K.box[1], v.y);
        I.z[a] = fmaf((float)sz, K.box[2], v.z);
        I.q[a] = K.epsfac * v.w;
        I.t[a] = A.type_slot[ci * 8 + a] * K.ntypes1 * 8;
    }
    float fi[24];
#pragma unroll
    for (int i = 0; i < 24; i++) fi[i] = 0.f;
    float elj = 0.f, ecoul = 0.f;
    __syncthreads();

    int2* q = s_q[warp];
    int2* m = s_m[warp];
    int nq = 0, mq = 0;
    const unsigned lt = (1u << lane) - 1u;
    unsigned bits = A.plane[(size_t)u.y * 8 + warp];
    unsigned ebits = A.plane_excl[(size_t)u.y * 8 + warp] & bits;
    int2 ent = ((bits >> lane) & 1u) ? A.jl[(size_t)u.y * 32 + lane] : make_int2(0, 0);
    for (int b = u.y; b < u.z; b++) {
        const bool last = b + 1 == u.z;
        unsigned bits_n = 0, ebits_n = 0;
        int2 ent_n = make_int2(0, 0);
        if (!last) {   // prefetch the next batch of the joint list
            bits_n = A.plane[(size_t)(b + 1) * 8 + warp];
            ebits_n = A.plane_excl[(size_t)(b + 1) * 8 + warp] & bits_n;
            if ((bits_n >> lane) & 1u) ent_n = A.jl[(size_t)(b + 1) * 32 + lane];
        }
        // compact the entries whose mask bit is set into the warp's two queues
        const unsigned nbits = bits & ~ebits;
        if ((nbits >> lane) & 1u) q[nq + __popc(nbits & lt)] = ent;
        if ((ebits >> lane) & 1u) m[mq + __popc(ebits & lt)] = ent;
        nq += __popc(nbits);
        mq += __popc(ebits);
        __syncwarp();
        // full unmasked steps; the j data of the next step is loaded before this step's arithmetic
        int done = 0;
        if (nq >= 4) {
            int cj = q[g].x;
            float4 xj = A.xq[cj * 8 + k];
            int tjb = A.type_slot[cj * 8 + k] * 8;
            while (true) {
                done += 4;
                const bool more = nq - done >= 4;
                int cj_n = cj;
                float4 xj_n = xj;
                int tjb_n = tjb;
                if (more) {
                    cj_n = q[done + g].x;
                    xj_n = A.xq[cj_n * 8 + k];
                    tjb_n = A.type_slot[cj_n * 8 + k] * 8;
                }
                float fjx, fjy, fjz;
                pair_step<COUL, ENERGY, false>(K, s_ljb, I, fi, elj, ecoul, xj, tjb, 0xffu, 0xffu, fjx, fjy, fjz);
                red_add_v4(&A.f4[cj * 8 + k], fjx, fjy, fjz);
                if (!more) break;
                cj = cj_n;
                xj = xj_n;
                tjb = tjb_n;
            }
        }
        const int rem = nq - done;
        int2 t = make_int2(0, 0);
        if (lane < rem) t = q[done + lane];
        __syncwarp();
        if (last) {   // the unit's tail goes through the masked queue (partly filled step allowed there)
            if (lane < rem) m[mq + lane] = t;
            mq += rem;
            nq = 0;
        } else {
            if (lane < rem) q[lane] = t;
            nq = rem;
        }
        __syncwarp();
        int md = 0;
        while (mq - md >= 4 || (last && mq - md > 0)) {
            const bool valid = g < mq - md;
            const int2 ce = valid ? m[md + g] : make_int2(ci, 0);
            const float4 xj = A.xq[ce.x * 8 + k];
            const int tjb = A.type_slot[ce.x * 8 + k] * 8;
            const ulonglong2 mm = *reinterpret_cast<const ulonglong2*>(&A.masks[((size_t)ce.y * 8 + warp) * 2]);
            const unsigned cbyte = valid ? (unsigned)(mm.y >> (8 * k)) & 0xffu : 0u;
            const unsigned mbyte = (unsigned)(mm.x >> (8 * k)) & cbyte;
            float fjx, fjy, fjz;
            pair_step<COUL, ENERGY, true>(K, s_ljb, I, fi, elj, ecoul, xj, tjb, cbyte, mbyte, fjx, fjy, fjz);
            if (valid) red_add_v4(&A.f4[ce.x * 8 + k], fjx, fjy, fjz);
            md += 4;
        }
        if (!last) {
            const int mrem = mq - md;
            int2 tm = make_int2(0, 0);
            if (lane < mrem) tm = m[md + lane];
            __syncwarp();
            if (lane < mrem) m[lane] = tm;
            __syncwarp();
            mq = mrem;
        }
        bits = bits_n;
        ebits = ebits_n;
        ent = ent_n;
    }

    if (ENERGY) {
        // per-shift sum of i forces for the virial (reading A8) and the energies, fp64 atomics per warp
        float sxs = 0.f, sys = 0.f, szs = 0.f;
#pragma unroll
        for (int a = 0; a < 8; a++) { sxs += fi[3 * a]; sys += fi[3 * a + 1]; szs += fi[3 * a + 2]; }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            sxs += __shfl_xor_sync(0xffffffffu, sxs, d);
            sys += __shfl_xor_sync(0xffffffffu, sys, d);
            szs += __shfl_xor_sync(0xffffffffu, szs, d);
            elj += __shfl_xor_sync(0xffffffffu, elj, d);
            ecoul += __shfl_xor_sync(0xffffffffu, ecoul, d);
        }
        if (lane == 0) {
            if (sid != NB_SHIFT_CENTER) {
                atomicAdd(&A.fshift[sid * 3 + 0], (double)sxs);
                atomicAdd(&A.fshift[sid * 3 + 1], (double)sys);
                atomicAdd(&A.fshift[sid * 3 + 2], (double)szs);
            }
            atomicAdd(&A.energies[0], (double)elj);
            atomicAdd(&A.energies[1], (double)ecoul);
        }
    }

    // (a8) i-force reduction: butterfly reduce-scatter of the 24 partial sums over the 32 lanes;
    // afterwards the quad lane>>2 == a holds (fx,fy,fz) of i atom a.
#pragma unroll
    for (int half = 12, d = 16; half >= 3; half >>= 1, d >>= 1) {
        const bool upper = (lane & d) != 0;
#pragma unroll
        for (int i = 0; i < half; i++) {
            const float keep = upper ? fi[i + half] : fi[i];
            const float send = upper ? fi[i] : fi[i + half];
            fi[i] = keep + __shfl_xor_sync(0xffffffffu, send, d);
        }
    }
#pragma unroll
    for (int d = 2; d > 0; d >>= 1) {
        fi[0] += __shfl_xor_sync(0xffffffffu, fi[0], d);
        fi[1] += __shfl_xor_sync(0xffffffffu, fi[1], d);
        fi[2] += __shfl_xor_sync(0xffffffffu, fi[2], d);
    }
    if ((lane & 3) == 0) red_add_v4(&A.f4[ci * 8 + (lane >> 2)], fi[0], fi[1], fi[2]);
}

// (a8) gather to the caller's atom order; leaves the accumulator zeroed for the next call.
template <bool VIRIAL>
__global__ void __launch_bounds__(256) k_gather(int nslots, float4* __restrict__ f4, const int* __restrict__ atom_of_slot,
                                                const float4* __restrict__ xq, float* __restrict__ f,
                                                double* __restrict__ xf /* [9] sum x (x) f */)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    double v[9];
#pragma unroll
    for (int i = 0; i < 9; i++) v[i] = 0.0;
    if (s < nslots) {
        const float4 fv = f4[s];
        f4[s] = make_float4(0.f, 0.f, 0.f, 0.f);
        const int a = atom_of_slot[s];
        if (a >= 0) {
            f[3 * a] = fv.x;
            f[3 * a + 1] = fv.y;
            f[3 * a + 2] = fv.z;
            if (VIRIAL) {
                const float4 x = xq[s];
                const double xx[3] = {x.x, x.y, x.z}, ff[3] = {fv.x, fv.y, fv.z};
#pragma unroll
                for (int l = 0; l < 3; l++)
#pragma unroll
                    for (int m = 0; m < 3; m++) v[3 * l + m] = xx[l] * ff[m];
            }
        }
    }
    if (VIRIAL) {
        __shared__ double s_v[8][9];
#pragma unroll
        for (int i = 0; i < 9; i++)
            for (int d = 16; d > 0; d >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], d);
        if ((threadIdx.x & 31) == 0)
            for (int i = 0; i < 9; i++) s_v[threadIdx.x >> 5][i] = v[i];
        __syncthreads();
        if (threadIdx.x < 9) {
            double t = 0.0;
            for (int w = 0; w < 8; w++) t += s_v[w][threadIdx.x];
            atomicAdd(&xf[threadIdx.x], t);
        }
    }
}

// Xi = -1/2 ( sum_i x_i (x) f_i + sum_s (s L) (x) S_s )   (reading A8)
__global__ void k_virial_final(const double* __restrict__ xf, const double* __restrict__ fshift, float3 box,
                               double* __restrict__ virial)
{
    const int i = threadIdx.x;
    if (i >= 9) return;
    const int l = i / 3, m = i % 3;
    double t = xf[i];
    const double L[3] = {box.x, box.y, box.z};
    for (int sid = 0; sid < NB_NSHIFT; sid++) {
        int s[3];
        nb_shift_vec(sid, s[0], s[1], s[2]);
        t += s[l] * L[l] * fshift[sid * 3 + m];
    }
    virial[i] = -0.5 * t;
}

__global__ void __launch_bounds__(256) k_fp32_peak(float* out, int iters, float a, float b)
{
    float x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}

// Counts atom pairs with r^2 < rc^2 over the inner list: interacting ("effective" pairs,
// PAPER.md L167-L173) and excluded-but-counted.  Same block/warp/lane mapping as the prune kernel.
__global__ void __launch_bounds__(256) k_count_pairs(ForceArgs A, unsigned long long* __restrict__ out)
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
        xi[a] = fmaf((float)sx, A.kc.box[0], v.x);
        yi[a] = fmaf((float)sy, A.kc.box[1], v.y);
        zi[a] = fmaf((float)sz, A.kc.box[2], v.z);
    }
    unsigned n_int = 0, n_exc = 0;
    for (int b = u.y; b < u.z; b++) {
        unsigned bits = A.plane[(size_t)b * 8 + warp];
        while (bits) {
            int my = -1;
#pragma unroll
            for (int t = 0; t < 4; t++) {
                const int p = bits ? __ffs(bits) - 1 : -1;
                bits &= bits - 1;
                if (t == g) my = p;
            }
            if (my < 0) continue;
            const int2 ce = A.jl[(size_t)b * 32 + my];
            const float4 xj = A.xq[ce.x * 8 + k];
            const ulonglong2 mm = *reinterpret_cast<const ulonglong2*>(&A.masks[((size_t)ce.y * 8 + warp) * 2]);
            const unsigned cbyte = (unsigned)(mm.y >> (8 * k)) & 0xffu, mbyte = (unsigned)(mm.x >> (8 * k)) & cbyte;
#pragma unroll
            for (int a = 0; a < 8; a++) {
                const float dx = xi[a] - xj.x, dy = yi[a] - xj.y, dz = zi[a] - xj.z;
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                if (r2 < A.kc.rc2) {
                    n_int += (mbyte >> a) & 1u;
                    n_exc += ((cbyte & ~mbyte) >> a) & 1u;
                }
            }
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        n_int += __shfl_xor_sync(0xffffffffu, n_int, d);
        n_exc += __shfl_xor_sync(0xffffffffu, n_exc, d);
    }
    if (lane == 0) {
        if (n_int) atomicAdd(&out[0], (unsigned long long)n_int);
        if (n_exc) atomicAdd(&out[1], (unsigned long long)n_exc);
    }
}

template <int COUL, bool ENERGY>
int launch_force(nb_ctx* c, const ForceArgs& A)
{
    const size_t smem = sizeof(float2) * (size_t)c->kc.ntypes1 * c->kc.ntypes1;
    static bool attr_set = false;
    if (!attr_set || smem > 48 * 1024) {
        NB_CUDA(c, cudaFuncSetAttribute(k_force<COUL, ENERGY>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
        attr_set = true;
    }
    k_force<COUL, ENERGY><<<c->nunits, 256, smem, c->stream>>>(A);
    NB_LAUNCH_CHECK(c);
    return NB_OK;
}

}  // namespace

int nbi_forces(nb_ctx* c, float* f, double* energies, double* virial)
{
    cudaStream_t st = c->stream;
    ForceArgs A;
    A.units = c->units_sorted.p;
    A.jl = c->jl.p;
    A.plane = c->plane_inner.p;
    A.plane_excl = c->plane_excl.p;
    A.xq = c->xq.p;
    A.type_slot = c->type_slot.p;
    A.ljtab = c->ljtab.p;
    A.masks = c->excl_masks.p;
    A.f4 = c->f4.p;
    A.kc = c->kc;
    for (int k = 0; k < 3; k++) A.kc.box[k] = c->box[k];
    {
        const float P[6] = {NB_EWC_P0, NB_EWC_P1, NB_EWC_P2, NB_EWC_P3, NB_EWC_P4, NB_EWC_P5};
        for (int k = 0; k < 6; k++) A.kc.ewp[k] = (float)((double)c->kc.beta3 * (double)P[k]);
    }
    NB_CUDA(c, c->fshift.ensure(NB_NSHIFT * 3 + 9, st));
    A.fshift = c->fshift.p;
    A.energies = energies;
    const bool energy = energies != nullptr;
    if (energy) {
        NB_CUDA(c, cudaMemsetAsync(energies, 0, 2 * sizeof(double), st));
        NB_CUDA(c, cudaMemsetAsync(c->fshift.p, 0, (NB_NSHIFT * 3 + 9) * sizeof(double), st));
    }
    int rc = NB_OK;
    if (c->nunits > 0) {
        NbStageTimer tm(c, NB_T_FORCE);
        if (c->prm.coulomb == NB_COUL_EWALD)
            rc = energy ? launch_force<NB_COUL_EWALD, true>(c, A) : launch_force<NB_COUL_EWALD, false>(c, A);
        else
            rc = energy ? launch_force<NB_COUL_RF, true>(c, A) : launch_force<NB_COUL_RF, false>(c, A);
        if (rc != NB_OK) return rc;
    }
    double* xf = c->fshift.p + NB_NSHIFT * 3;
    const int nb = (c->nslots + 255) / 256;
    NbStageTimer tm(c, NB_T_REDUCE);
    if (virial)
        k_gather<true><<<nb, 256, 0, st>>>(c->nslots, c->f4.p, c->atom_of_slot.p, c->xq.p, f, xf);
    else
        k_gather<false><<<nb, 256, 0, st>>>(c->nslots, c->f4.p, c->atom_of_slot.p, c->xq.p, f, xf);
    NB_LAUNCH_CHECK(c);
    if (virial) {
        k_virial_final<<<1, 32, 0, st>>>(xf, c->fshift.p, make_float3(c->box[0], c->box[1], c->box[2]), virial);
        NB_LAUNCH_CHECK(c);
    }
    c->st.force_count++;
    return NB_OK;
}

int nbi_measure_fp32_peak(nb_ctx* c, double* fma_per_s)
{
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, c->prm.device);
    const int grid = nsm * 8, iters = 4000;
    DevBuf<float> out;
    NB_CUDA(c, out.ensure((size_t)grid * 256, c->stream));
    cudaEvent_t e0, e1;
    NB_CUDA(c, cudaEventCreate(&e0));
    NB_CUDA(c, cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 5; rep++) {
        cudaEventRecord(e0, c->stream);
        k_fp32_peak<<<grid, 256, 0, c->stream>>>(out.p, iters, 1.0001f, 0.5f);
        cudaEventRecord(e1, c->stream);
        NB_CUDA(c, cudaEventSynchronize(e1));
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    out.release();
    *fma_per_s = (double)grid * 256 * iters * 64.0 / (best * 1e-3);
    return NB_OK;
}

int nbi_count_pairs(nb_ctx* c, int64_t* n_interacting, int64_t* n_excluded)
{
    cudaStream_t st = c->stream;
    ForceArgs A;
    memset(&A, 0, sizeof(A));
    A.units = c->units_canon.p;
    A.jl = c->jl.p;
    A.plane = c->plane_inner.p;
    A.xq = c->xq.p;
    A.masks = c->excl_masks.p;
    A.kc = c->kc;
    for (int k = 0; k < 3; k++) A.kc.box[k] = c->box[k];
    NB_CUDA(c, c->counters.ensure(8, st));
    NB_CUDA(c, cudaMemsetAsync(c->counters.p, 0, 8 * sizeof(long long), st));
    if (c->nunits > 0) {
        k_count_pairs<<<c->nunits, 256, 0, st>>>(A, (unsigned long long*)c->counters.p);
        NB_LAUNCH_CHECK(c);
    }
    long long v[2] = {0, 0};
    NB_CUDA(c, cudaMemcpyAsync(v, c->counters.p, sizeof(v), cudaMemcpyDeviceToHost, st));
    NB_CUDA(c, cudaStreamSynchronize(st));
    if (n_interacting) *n_interacting = v[0];
    if (n_excluded) *n_excluded = v[1];
    return NB_OK;
}
