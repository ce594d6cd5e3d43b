// ris_grad_kernel.cuh -- the fused class kernel: S1 Boys + S2 derivative-integral recurrence +
// S3 contraction with the D / Gamma^P tile + S4 reduction, one instantiation per
// (l_mu,l_nu) class.  Eq. 27 terms 1-2 for the integrals of Eq. 21
// (PAPER.md:119).
//
// Mapping ("aux lanes"): the 32 lanes of a warp hold 32 different auxiliary functions P (blockIdx.y selects the
// chunk of 32) and walk TOGETHER through the shell pairs of a warp task (a window of ~64 packed primitive pairs,
// ris_internal.h).  Everything that belongs to the shell pair -- pair record, primitive-pair records, loop trip counts,
// the host-centre phases, the D tile of the J term -- is therefore warp-uniform: it is staged once per task into the
// warp's shared memory with coalesced 16-byte copies and read back as broadcasts, there is no divergence except the
// Boys-function branch, and what varies per lane (aux centre / exponent, W - P, Boys values, the Gamma^P tile of the
// K term, stored P-minor so a warp reads 256 contiguous bytes) is exactly the per-lane arithmetic.
// The per-state gradient accumulators are per-lane shared-memory slots (conflict-free: lane-contiguous), which keeps the
// register file for the recurrence and lets the light classes run 16 warps per SM:
//   aux side   g[A_P] = -(dA + dB) summed over the pairs (translational invariance): the lane owns P, so this is one
//              slot per (state, x) over ALL tasks of the warp; the four warps of a block (same P chunk) are summed
//              in fixed order at the end, one atomic per (block, P, state, x).
//   pair side  g[A_mu], g[A_nu]: slots across the consecutive shell pairs of one atom pair (the pairs of a class
//              are sorted by atom pair), then a fixed-order sum over the lanes and one atomic per (atom pair, state,
//              centre, x).
// Every in-block sum has a fixed order; the global atomics are FP64 adds, or -- deterministic mode -- 64-bit integer
// adds of a fixed-point split (ris_grad_add), which makes the result bitwise reproducible.
#pragma once
#include "ris_core.cuh"
#include "ris_internal.h"

// One host-centre phase of a contracted triplet: the primitive pairs q[0 .. nk) hosted on centre Z (host l = LH,
// other l = LO), then HRR / derivative / tile contraction into the lane's accumulator slots.
template <int LH, int LO, bool TR>
RIS_DEV void ris_phase(int nk, const double* __restrict__ q, double ZCx, double ZCy, double ZCz, double ZOx, double ZOy,
                       double ZOz, double alpha, double auxfac, const double* __restrict__ boys,
                       const double* __restrict__ tile, size_t estride, size_t sstride, int nb, const double* __restrict__ sc,
                       double* __restrict__ slot)
{
    using K = RisClass<LH, LO>;
    double acc[K::NACC];
#pragma unroll
    for (int i = 0; i < K::NACC; ++i) acc[i] = 0.0;
    for (int k = 0; k < nk; ++k, q += RIS_PRIM_FIELDS) {
        const double2 r0 = *reinterpret_cast<const double2*>(q);
        const double2 r1 = *reinterpret_cast<const double2*>(q + 2);
        const double2 r2 = *reinterpret_cast<const double2*>(q + 4);
        const double2 r3 = *reinterpret_cast<const double2*>(q + 6);
        ris_prim_triplet<LH, LO>(r0.x, r0.y, r1.x, r1.y, r2.x, TR ? r3.x : r2.y, TR ? r2.y : r3.x, r3.y, ZCx, ZCy, ZCz,
                                 alpha, auxfac, boys, acc);
    }
    ris_hrrc<LH, LO, TR, 33, 32>(acc, ZOx, ZOy, ZOz, tile, estride, sstride, nb, sc, slot);
}

template <int NEL>
RIS_DEV void ris_prefetch_tile(const double* t, size_t estride, size_t sstride, int nb, int lstride)
{
    const int rows = lstride ? NEL : (NEL + 15) / 16;
    const size_t step = lstride ? estride : 16;
    for (int s = 0; s < nb; ++s)
        for (int e = 0; e < rows; ++e) asm volatile("prefetch.global.L1 [%0];" ::"l"(t + (size_t)s * sstride + (size_t)e * step));
}

// resident blocks per SM the register allocation aims at (light classes: latency-bound prefactor / Boys chains
// want warps; heavy classes: the contracted targets want registers)
#ifndef RIS_MB1
#define RIS_MB1 4
#define RIS_MB2 3
#define RIS_MB3 2
#define RIS_MB4 2
#endif
// SPLIT: the heavy classes (l_mu + l_nu >= 4) run their two host-centre phases as two launches (PH = 1: primitive pairs
// hosted on A, PH = 2: hosted on B; PH = 0: both in one kernel).  With both phases inlined the (2,2) kernel is 94 KB of
// SASS and stalls on instruction fetch (profiles/r01_v5_ncu.md: no_instruction 7.1 cycles per issue); one phase is 47 KB.
#ifndef RIS_SPLIT_L
#define RIS_SPLIT_L 4
#endif
template <int LA, int LB> struct RisGradTune {
    static constexpr int MINB = (LA + LB <= 1) ? RIS_MB1 : (LA + LB == 2 ? RIS_MB2 : (LA + LB == 3 ? RIS_MB3 : RIS_MB4));
    static constexpr bool SPLIT = (LA + LB >= RIS_SPLIT_L);
};

template <int LA, int LB, int PH>
__global__ void __launch_bounds__(RIS_GRAD_THREADS, RisGradTune<LA, LB>::MINB) ris_grad_kernel(const RisGradParams prm)
{
    constexpr int NEL = RisClass<LA, LB>::NCA * RisClass<LA, LB>::NCB;
    extern __shared__ __align__(16) unsigned char sm_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const RisClassPack& pk = prm.pk;
    const int nb = prm.nb;
    const size_t wbytes = ris_grad_warp_smem(pk.kmax, nb);
    double* s_prim = reinterpret_cast<double*>(sm_raw + (size_t)warp * wbytes);
    RisPairRec* s_pair = reinterpret_cast<RisPairRec*>(s_prim + (size_t)RIS_PRIM_FIELDS * (RIS_TASK_PRIMS + pk.kmax));
    double* s_red = reinterpret_cast<double*>(s_pair + RIS_TASK_PRIMS);      // [6 nb][33]  pair side: A x,y,z, B x,y,z per state
    double* s_gaux = s_red + 6 * nb * 33;                                    // [3 nb][32]  aux side
    double* s_sc = s_gaux + 3 * nb * 32;                                     // [nb][32]    J: c_aux[s][P]; K: 1
    const size_t gaux_off = (size_t)(reinterpret_cast<unsigned char*>(s_gaux) - (sm_raw + (size_t)warp * wbytes));

    // this lane's auxiliary function
    const int P = prm.p0 + blockIdx.y * 32 + lane;
    const bool live = P < prm.p1;
    const int Pe = live ? P : prm.p1 - 1;
    const double* ax = prm.aux + 5 * (size_t)Pe;
    const double Cx = ax[0], Cy = ax[1], Cz = ax[2], alpha = ax[3];
    const double auxfac = live ? ax[4] : 0.0;          // a dead lane computes exact zeros
    for (int s = 0; s < nb; ++s) s_sc[s * 32 + lane] = prm.cscale ? prm.cscale[(size_t)s * prm.naux + Pe] : 1.0;
    for (int i = 0; i < 6 * nb; ++i) s_red[i * 33 + lane] = 0.0;
    for (int i = 0; i < 3 * nb; ++i) s_gaux[i * 32 + lane] = 0.0;
    const double* __restrict__ tile_lane = prm.tile + (size_t)(Pe - prm.p0) * prm.lstride;
    const size_t estride = (size_t)prm.estride, sstride = (size_t)prm.sstride;
    int curA = -1, curB = -1;
    __syncwarp();

    // pair side: fixed-order sum over the lanes, one atomic per (state, centre, x); aux side keeps -(gA + gB)
    auto flush = [&]() {
        if (curA < 0) return;
        for (int s = 0; s < nb; ++s)
#pragma unroll
            for (int x = 0; x < 3; ++x)
                s_gaux[(s * 3 + x) * 32 + lane] -= s_red[(s * 6 + x) * 33 + lane] + s_red[(s * 6 + 3 + x) * 33 + lane];
        __syncwarp();
        if (lane < 6 * nb) {
            const double* r = s_red + lane * 33;
            double v = 0.0;
#pragma unroll 8
            for (int j = 0; j < 32; ++j) v += r[j];
            const int s = lane / 6, c = lane - 6 * s;
            const int at = c < 3 ? curA : curB;
            ris_grad_add(prm, ((size_t)s * prm.natoms + at) * 3 + (c < 3 ? c : c - 3), v);
        }
        __syncwarp();
        for (int i = 0; i < 6 * nb; ++i) s_red[i * 33 + lane] = 0.0;
        __syncwarp();
    };

    // Tasks are handed out by an atomic ticket counter per aux chunk; the ticket for the NEXT task is drawn before the
    // current one starts, so its latency is hidden.  Every warp ends within one task of the others, and a block that
    // becomes resident late finds the counter exhausted and leaves.
    int task = 0;
    if (lane == 0) task = atomicAdd(prm.task_ctr + blockIdx.y, 1);
    task = __shfl_sync(0xffffffffu, task, 0);
    while (task < pk.ntasks) {
        int next = 0;
        if (lane == 0) next = atomicAdd(prm.task_ctr + blockIdx.y, 1);
        const int ip0 = pk.task_begin[task], ip1 = pk.task_begin[task + 1];
        const long long q0 = pk.prim_off[ip0], q1 = pk.prim_off[ip1];
        __syncwarp();
        {   // stage the task: 16-byte copies, 4 per record
            const int4* src = reinterpret_cast<const int4*>(pk.prim + (size_t)q0 * RIS_PRIM_FIELDS);
            int4* dst = reinterpret_cast<int4*>(s_prim);
            const int n = (int)(q1 - q0) * 4;
            for (int i = lane; i < n; i += 32) dst[i] = src[i];
            const int4* srcp = reinterpret_cast<const int4*>(pk.pairs + ip0);
            int4* dstp = reinterpret_cast<int4*>(s_pair);
            const int np4 = (ip1 - ip0) * 4;
            for (int i = lane; i < np4; i += 32) dstp[i] = srcp[i];
        }
        __syncwarp();
        const double* __restrict__ q = s_prim;
        for (int j = 0; j < ip1 - ip0; ++j) {
            const RisPairRec pr = s_pair[j];
            if (pr.atA != curA || pr.atB != curB) { flush(); curA = pr.atA; curB = pr.atB; }
            const double* __restrict__ tile = tile_lane + ((size_t)pk.elem_off + (size_t)(ip0 + j) * NEL) * estride;
            const double ACx = pr.Ax - Cx, ACy = pr.Ay - Cy, ACz = pr.Az - Cz;
#ifdef RIS_PREFETCH_TILE   // measured on config 4: no gain (7.6 -> 7.9 ms/step), kept for experiments
            // the NEXT pair's tile rows start their way from HBM / L2 to L1 while this pair's primitives run
            // (K: one 256-byte row per element and state across the warp; J: the pair's few contiguous lines)
            if (ip0 + j + 1 < pk.npairs) ris_prefetch_tile<NEL>(tile + (size_t)NEL * estride, estride, sstride, nb, prm.lstride);
#endif
            if (PH != 2 && pr.nkA > 0)
                ris_phase<LA, LB, false>(pr.nkA, q, ACx, ACy, ACz, pr.ABx, pr.ABy, pr.ABz, alpha, auxfac, prm.boys, tile,
                                         estride, sstride, nb, s_sc + lane, s_red + lane);
            q += (size_t)pr.nkA * RIS_PRIM_FIELDS;
            if (PH != 1 && pr.nkB > 0)
                ris_phase<LB, LA, true>(pr.nkB, q, ACx - pr.ABx, ACy - pr.ABy, ACz - pr.ABz, -pr.ABx, -pr.ABy, -pr.ABz, alpha,
                                        auxfac, prm.boys, tile, estride, sstride, nb, s_sc + lane, s_red + lane);
            q += (size_t)pr.nkB * RIS_PRIM_FIELDS;
        }
        if (prm.det != nullptr) {
            // deterministic mode: which warp runs which task varies from run to run, so every task hands over its own
            // sums (integer atomics: exact, order-independent) instead of carrying FP64 partial sums into the next task
            flush();
            curA = curB = -1;
            if (live)
                for (int i = 0; i < 3 * nb; ++i) {
                    ris_grad_add(prm, ((size_t)(i / 3) * prm.natoms + P) * 3 + (i % 3), s_gaux[i * 32 + lane]);
                    s_gaux[i * 32 + lane] = 0.0;
                }
        }
        task = __shfl_sync(0xffffffffu, next, 0);
    }
    flush();

    // aux side: the four warps of the block hold the same 32 aux functions
    __syncthreads();
    if (warp == 0 && live) {
        for (int i = 0; i < 3 * nb; ++i) {
            double v = 0.0;
#pragma unroll
            for (int w = 0; w < RIS_GRAD_WARPS; ++w)
                v += reinterpret_cast<const double*>(sm_raw + (size_t)w * wbytes + gaux_off)[i * 32 + lane];
            const int s = i / 3, x = i - 3 * s;
            ris_grad_add(prm, ((size_t)s * prm.natoms + P) * 3 + x, v);
        }
    }
}

template <int LA, int LB, int PH>
void ris_launch_grad_phase(const RisGradParams& p, cudaStream_t st)
{
    const size_t smem = RIS_GRAD_WARPS * ris_grad_warp_smem(p.pk.kmax, p.nb);
    static size_t configured = 0;
    if (smem > 48 * 1024 && smem > configured) {
        cudaFuncSetAttribute(ris_grad_kernel<LA, LB, PH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        configured = smem;
    }
    // blockIdx.y: chunks of 32 aux functions; blockIdx.x: the blocks of a chunk, together one resident wave of
    // long-lived warps drawing tasks (few aux-side atomics, no wave quantisation)
    const int ny = (p.p1 - p.p0 + 31) / 32;
    const int nbt = (p.pk.ntasks + RIS_GRAD_WARPS - 1) / RIS_GRAD_WARPS;
    static int nsm = 0;
    if (nsm == 0) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev); }
    const int nx = std::max(1, std::min(nbt, (nsm * RisGradTune<LA, LB>::MINB + ny - 1) / ny));
    ris_grad_kernel<LA, LB, PH><<<dim3(nx, ny), RIS_GRAD_THREADS, smem, st>>>(p);
}

// p.task_ctr holds two zeroed ticket arrays of ny counters each (one per phase launch)
template <int LA, int LB>
void ris_launch_grad(const RisGradParams& p, cudaStream_t st)
{
    if (p.pk.npairs <= 0 || p.pk.ntasks <= 0 || p.p1 <= p.p0) return;
    if constexpr (RisGradTune<LA, LB>::SPLIT) {
        RisGradParams q = p;
        ris_launch_grad_phase<LA, LB, 1>(q, st);
        q.task_ctr = p.task_ctr + (p.p1 - p.p0 + 31) / 32;
        ris_launch_grad_phase<LA, LB, 2>(q, st);
    } else {
        ris_launch_grad_phase<LA, LB, 0>(p, st);
    }
}
