// ris_grad_kernel.cuh -- the fused class kernel: S1 Boys + S2 derivative-integral recurrence +
// S3 contraction with the D / Gamma^P tile + S4 reduction, one instantiation per
// (l_mu,l_nu) class.  Eq. 27 terms 1-2 for the integrals of Eq. 21.
//
// Mapping: one thread = one packed shell pair of the class; the thread loops over the aux functions
// P of its blockIdx.y chunk, and for each P over the surviving primitive pairs (contraction in
// registers), then runs the contracted HRR / derivative / tile contraction for every state.
//   pair-side gradients g[A_mu], g[A_nu]: per-thread shared-memory slots across the whole P loop,
//       one global atomic per (thread, state, component) at the end;
//   aux-side gradient g[A_P] = -(g_mu + g_nu) (translational invariance): warp-shuffle reduction per
//       (P, state) into a per-warp shared-memory slot (no shared atomics), the warps' slots summed in fixed order
//       at the end, one global atomic per (block, P, state, x).
// Every in-block sum has a fixed order; the global atomics are FP64 adds, or -- deterministic mode -- 64-bit integer
// adds of a fixed-point split (ris_grad_add), which makes the result bitwise reproducible.
#pragma once
#include "ris_core.cuh"
#include "ris_internal.h"

RIS_DEV double ris_warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// One phase of a contracted triplet: the primitive pairs [k0, k1) hosted on centre Z (host l = LH, other
// l = LO), then HRR / derivative / tile contraction; `sink(s, g_host[3], g_other[3])` per state.
template <int LH, int LO, bool TR, class Sink>
RIS_DEV void ris_phase(int k0, int k1, const double* __restrict__ prim, size_t fs, double Zx, double Zy, double Zz,
                       double ZOx, double ZOy, double ZOz, double Cx, double Cy, double Cz, double alpha, double auxfac,
                       const double* __restrict__ boys, const double* __restrict__ tile, size_t sstride, int nb, Sink&& sink)
{
    using K = RisClass<LH, LO>;
    double acc[K::NACC];
#pragma unroll
    for (int i = 0; i < K::NACC; ++i) acc[i] = 0.0;
    const double ZCx = Zx - Cx, ZCy = Zy - Cy, ZCz = Zz - Cz;
    for (int k = k0; k < k1; ++k) {
        const double* __restrict__ q = prim + (size_t)k * RIS_PRIM_FIELDS * fs;
        const double a2 = q[5 * fs], b2 = q[6 * fs];
        ris_prim_triplet<LH, LO>(q[0], q[fs], q[2 * fs], q[3 * fs], q[4 * fs], TR ? b2 : a2, TR ? a2 : b2, q[7 * fs],
                                 ZCx, ZCy, ZCz, alpha, auxfac, boys, acc);
    }
    ris_hrrc<LH, LO, TR>(acc, Zx - ZOx, Zy - ZOy, Zz - ZOz, tile, fs, sstride, nb, sink);
}

template <int LA, int LB>
__global__ void __launch_bounds__(RIS_GRAD_THREADS) ris_grad_kernel(const RisGradParams prm)
{
    constexpr int NT = RIS_GRAD_THREADS;
    extern __shared__ double sm[];
    const int tid = threadIdx.x;
    const int nb = prm.nb;
    const int pc0 = prm.p0 + blockIdx.y * prm.pchunk;
    const int npc = min(pc0 + prm.pchunk, prm.p1) - pc0;
    double* s_aux = sm;                              // [pchunk][5]
    constexpr int NW = NT / 32;
    double* s_gaux = s_aux + 5 * prm.pchunk;         // [NW][pchunk][nb][3]   per-warp aux-side accumulators
    double* s_slot = s_gaux + 3 * nb * prm.pchunk * NW;   // [nb][6][NT]  pair-side accumulators (A: 0..2, B: 3..5)
    double* s_stash = s_slot + 6 * nb * NT;          // [nb][3][NT]  dA+dB of the current contracted triplet
    for (int i = tid; i < 5 * npc; i += NT) s_aux[i] = prm.aux[5 * (size_t)pc0 + i];
    for (int i = tid; i < 3 * nb * prm.pchunk * NW; i += NT) s_gaux[i] = 0.0;
    for (int i = 0; i < 6 * nb; ++i) s_slot[i * NT + tid] = 0.0;
    __syncthreads();

    const RisClassPack& pk = prm.pk;
    const int npad = pk.npad;
    const int ip = blockIdx.x * NT + tid;
    const bool active = ip < pk.npairs;
    const size_t fs = (size_t)npad;                  // field stride
    const double Ax = pk.geom[0 * fs + ip], Ay = pk.geom[1 * fs + ip], Az = pk.geom[2 * fs + ip];
    const double Bx = Ax - pk.geom[3 * fs + ip], By = Ay - pk.geom[4 * fs + ip], Bz = Az - pk.geom[5 * fs + ip];
    const int nkA = active ? pk.nkA[ip] : 0;
    const int nk = nkA + (active ? pk.nkB[ip] : 0);
    // a phase is skipped only when no lane of the warp needs it (the sink contains warp shuffles)
    const bool doA = __any_sync(0xffffffffu, nkA > 0), doB = __any_sync(0xffffffffu, nk > nkA);
    const double* __restrict__ prim = pk.prim + ip;

    for (int pl = 0; pl < npc; ++pl) {
        const double Cx = s_aux[5 * pl + 0], Cy = s_aux[5 * pl + 1], Cz = s_aux[5 * pl + 2];
        const double alpha = s_aux[5 * pl + 3], auxfac = s_aux[5 * pl + 4];
        const int P = pc0 + pl;
        const double* __restrict__ tile = prm.tile + (size_t)(P - prm.p0) * prm.pstride + pk.elem_off + ip;
        for (int s = 0; s < 3 * nb; ++s) s_stash[s * NT + tid] = 0.0;
        // gA / gB of state s, scaled; accumulates the pair side and stashes dA + dB
        auto add = [&](int s, double a0, double a1, double a2, double b0, double b1, double b2) {
            double sc = prm.cscale ? prm.cscale[(size_t)s * prm.naux + P] : 1.0;
            if (!active) { sc = 0.0; a0 = a1 = a2 = b0 = b1 = b2 = 0.0; }
            a0 *= sc; a1 *= sc; a2 *= sc; b0 *= sc; b1 *= sc; b2 *= sc;
            double* sl = s_slot + (size_t)s * 6 * NT + tid;
            sl[0 * NT] += a0; sl[1 * NT] += a1; sl[2 * NT] += a2;
            sl[3 * NT] += b0; sl[4 * NT] += b1; sl[5 * NT] += b2;
            double* st = s_stash + (size_t)s * 3 * NT + tid;
            st[0 * NT] += a0 + b0; st[1 * NT] += a1 + b1; st[2 * NT] += a2 + b2;
        };
        if (doA)
            ris_phase<LA, LB, false>(0, nkA, prim, fs, Ax, Ay, Az, Bx, By, Bz, Cx, Cy, Cz, alpha, auxfac, prm.boys, tile,
                                     (size_t)prm.sstride, nb,
                                     [&](int s, double h0, double h1, double h2, double o0, double o1, double o2) {
                                         add(s, h0, h1, h2, o0, o1, o2);
                                     });
        if (doB)
            ris_phase<LB, LA, true>(nkA, nk, prim, fs, Bx, By, Bz, Ax, Ay, Az, Cx, Cy, Cz, alpha, auxfac, prm.boys, tile,
                                    (size_t)prm.sstride, nb,
                                    [&](int s, double h0, double h1, double h2, double o0, double o1, double o2) {
                                        add(s, o0, o1, o2, h0, h1, h2);
                                    });
        // aux side: g[A_P] -= sum over the warp's pairs of (dA + dB)   (translational invariance)
        for (int s = 0; s < nb; ++s) {
            const double* st = s_stash + (size_t)s * 3 * NT + tid;
            const double t0 = ris_warp_sum(st[0 * NT]), t1 = ris_warp_sum(st[1 * NT]), t2 = ris_warp_sum(st[2 * NT]);
            if ((tid & 31) == 0) {
                double* g = s_gaux + (((size_t)(tid >> 5) * prm.pchunk + pl) * nb + s) * 3;
                g[0] -= t0; g[1] -= t1; g[2] -= t2;
            }
        }
    }
    __syncthreads();
    if (active) {
        const int atA = pk.atoms[ip], atB = pk.atoms[(size_t)npad + ip];
        for (int s = 0; s < nb; ++s) {
            const double* sl = s_slot + (size_t)s * 6 * NT + tid;
            const size_t iA = ((size_t)s * prm.natoms + atA) * 3, iB = ((size_t)s * prm.natoms + atB) * 3;
            ris_grad_add(prm, iA + 0, sl[0 * NT]); ris_grad_add(prm, iA + 1, sl[1 * NT]); ris_grad_add(prm, iA + 2, sl[2 * NT]);
            ris_grad_add(prm, iB + 0, sl[3 * NT]); ris_grad_add(prm, iB + 1, sl[4 * NT]); ris_grad_add(prm, iB + 2, sl[5 * NT]);
        }
    }
    for (int i = tid; i < 3 * nb * npc; i += NT) {
        const int pl = i / (3 * nb), r = i - pl * 3 * nb, s = r / 3, x = r - 3 * s;
        double v = 0.0;
        for (int w = 0; w < NW; ++w) v += s_gaux[(size_t)w * 3 * nb * prm.pchunk + i];
        ris_grad_add(prm, ((size_t)s * prm.natoms + (pc0 + pl)) * 3 + x, v);
    }
}

inline size_t ris_grad_smem_bytes(const RisGradParams& p)
{
    return sizeof(double) * ((size_t)5 * p.pchunk + (size_t)3 * p.nb * p.pchunk * (RIS_GRAD_THREADS / 32) + (size_t)9 * p.nb * RIS_GRAD_THREADS);
}

template <int LA, int LB>
void ris_launch_grad(const RisGradParams& p, cudaStream_t st)
{
    if (p.pk.npairs <= 0 || p.p1 <= p.p0) return;
    const size_t smem = ris_grad_smem_bytes(p);
    static size_t configured = 0;
    if (smem > 48 * 1024 && smem > configured) {
        cudaFuncSetAttribute(ris_grad_kernel<LA, LB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        configured = smem;
    }
    dim3 grid(p.pk.npad / RIS_GRAD_THREADS, (p.p1 - p.p0 + p.pchunk - 1) / p.pchunk);
    ris_grad_kernel<LA, LB><<<grid, RIS_GRAD_THREADS, smem, st>>>(p);
}
