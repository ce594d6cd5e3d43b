// ris_int_kernel.cuh -- the undifferentiated class kernel of the fitting step:
//   v[s][P] = sum_{mu nu} D^s_{mu nu} (mu nu|P)             (first factor of Eq. 21)
// Same mapping as ris_grad_kernel ("aux lanes": a warp's 32 lanes hold 32 aux functions P and walk together through
// the shell pairs of a warp task; pair data warp-uniform, staged in shared memory), same packed pair records, same
// folded tile (D + D^T on unique pairs, 1/2 on the shell diagonal), same two host-centre phases.  The recurrence
// stops one level lower (e <= l_mu + l_nu) and there is nothing to reduce over atoms: the lane owns P, so v[s][P] is a
// per-lane sum over ALL shell pairs; the four warps of a block are added in fixed order and leave one atomic per
// (block, P, state).
#pragma once
#include "ris_core.cuh"
#include "ris_internal.h"

// STORE: instead of the dot with a tile, the contracted integrals themselves are added to out[el * ostride] (the
// P-minor integral buffer of ris_fit_K); tile / slot are unused then.
template <int LH, int LO, bool TR, bool STORE, int AUX>
RIS_DEV void ris_phase0(int nk, const double* __restrict__ q, double ZCx, double ZCy, double ZCz, double ZOx, double ZOy,
                        double ZOz, double alpha, double auxfac, const double* __restrict__ boys,
                        const double* __restrict__ tile, size_t sstride, int nb, double* __restrict__ slot,
                        double* __restrict__ out, size_t ostride)
{
    using K = RisClass0<LH, LO>;
    double acc[K::NACC];
#pragma unroll
    for (int i = 0; i < K::NACC; ++i) acc[i] = 0.0;
    for (int k = 0; k < nk; ++k, q += RIS_PRIM_FIELDS) {
        const double2 r0 = *reinterpret_cast<const double2*>(q);
        const double2 r1 = *reinterpret_cast<const double2*>(q + 2);
        const double2 r2 = *reinterpret_cast<const double2*>(q + 4);
        const double2 r3 = *reinterpret_cast<const double2*>(q + 6);
        if constexpr (AUX == 0) ris_prim_triplet0<LH, LO>(r0.x, r0.y, r1.x, r1.y, r2.x, r3.y, ZCx, ZCy, ZCz, alpha, auxfac, boys, acc);
        else ris_prim_triplet0_p<LH, LO, AUX - 1>(r0.x, r0.y, r1.x, r1.y, r2.x, r3.y, ZCx, ZCy, ZCz, alpha, auxfac, boys, acc);
    }
    if constexpr (STORE) ris_hrr0w<LH, LO, TR>(acc, ZOx, ZOy, ZOz, out, ostride);
    else ris_hrr0c<LH, LO, TR, 32>(acc, ZOx, ZOy, ZOz, tile, (size_t)1, sstride, nb, slot);
}

// dynamic shared memory per warp: the task's primitive-pair and pair records + [nb][32] sums
__host__ __device__ inline size_t ris_int_warp_smem(int kmax, int nb)
{
    return (size_t)64 * (RIS_TASK_PRIMS + kmax) + (size_t)64 * RIS_TASK_PRIMS + (size_t)8 * nb * 32;
}

// prm.tile: J tile [nb][packed elements] (estride 1); prm.grad: v [nb][naux] (zeroed by the caller).
// STORE: prm.grad is the integral buffer [packed elements][estride] (function-minor, zeroed by the caller), element el of
// the auxiliary function with index fn (its record's id) at grad[el * estride + fn]; nb is 0.
template <int LA, int LB, bool STORE, int AUX = 0>
__global__ void __launch_bounds__(RIS_GRAD_THREADS, 3) ris_int_kernel(const RisGradParams prm)
{
    constexpr int NEL = RisClass<LA, LB>::NCA * RisClass<LA, LB>::NCB;
    extern __shared__ __align__(16) unsigned char sm_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const RisClassPack& pk = prm.pk;
    const int nb = prm.nb;
    const size_t wbytes = ris_int_warp_smem(pk.kmax, nb);
    double* s_prim = reinterpret_cast<double*>(sm_raw + (size_t)warp * wbytes);
    RisPairRec* s_pair = reinterpret_cast<RisPairRec*>(s_prim + (size_t)RIS_PRIM_FIELDS * (RIS_TASK_PRIMS + pk.kmax));
    double* s_v = reinterpret_cast<double*>(s_pair + RIS_TASK_PRIMS);       // [nb][32]
    const size_t v_off = (size_t)(reinterpret_cast<unsigned char*>(s_v) - (sm_raw + (size_t)warp * wbytes));

    const int pos = prm.p0 + blockIdx.y * 32 + lane;       // position in the launch's list of auxiliary functions
    const bool live = pos < prm.p1;
    const int Pe = live ? pos : prm.p1 - 1;
    const double* ax = prm.aux + RIS_AUX_FIELDS * (size_t)Pe;
    const double Cx = ax[0], Cy = ax[1], Cz = ax[2], alpha = ax[3];
    const double auxfac = live ? ax[4] : 0.0;
    const int fn = reinterpret_cast<const int2*>(ax + 5)->y;  // index of the function: its entry of v
    for (int s = 0; s < nb; ++s) s_v[s * 32 + lane] = 0.0;
    const size_t sstride = (size_t)prm.sstride;
    __syncwarp();

    int task = 0;
    if (lane == 0) task = atomicAdd(prm.task_ctr + blockIdx.y, 1);
    task = __shfl_sync(0xffffffffu, task, 0);
    while (task < pk.ntasks) {
        int next = 0;
        if (lane == 0) next = atomicAdd(prm.task_ctr + blockIdx.y, 1);
        const int ip0 = pk.task_begin[task], ip1 = pk.task_begin[task + 1];
        const long long q0 = pk.prim_off[ip0], q1 = pk.prim_off[ip1];
        __syncwarp();
        {
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
            const double* __restrict__ tile = STORE ? nullptr : prm.tile + (size_t)pk.elem_off + (size_t)(ip0 + j) * NEL;
            // a dead lane (P beyond the range) must not write: the phases below are skipped for it
            double* __restrict__ out = STORE ? prm.grad + ((size_t)pk.elem_off + (size_t)(ip0 + j) * NEL) * (size_t)prm.estride + fn
                                            : nullptr;
            const double ACx = pr.Ax - Cx, ACy = pr.Ay - Cy, ACz = pr.Az - Cz;
            if (pr.nkA > 0 && (!STORE || live))
                ris_phase0<LA, LB, false, STORE, AUX>(pr.nkA, q, ACx, ACy, ACz, pr.ABx, pr.ABy, pr.ABz, alpha, auxfac, prm.boys, tile,
                                                 sstride, nb, s_v + lane, out, (size_t)prm.estride);
            q += (size_t)pr.nkA * RIS_PRIM_FIELDS;
            if (pr.nkB > 0 && (!STORE || live))
                ris_phase0<LB, LA, true, STORE, AUX>(pr.nkB, q, ACx - pr.ABx, ACy - pr.ABy, ACz - pr.ABz, -pr.ABx, -pr.ABy, -pr.ABz,
                                                alpha, auxfac, prm.boys, tile, sstride, nb, s_v + lane, out, (size_t)prm.estride);
            q += (size_t)pr.nkB * RIS_PRIM_FIELDS;
        }
        task = __shfl_sync(0xffffffffu, next, 0);
    }
    __syncthreads();
    if (!STORE && warp == 0 && live) {
        for (int s = 0; s < nb; ++s) {
            double v = 0.0;
#pragma unroll
            for (int w = 0; w < RIS_GRAD_WARPS; ++w)
                v += reinterpret_cast<const double*>(sm_raw + (size_t)w * wbytes + v_off)[s * 32 + lane];
            atomicAdd(prm.grad + (size_t)s * prm.naux + fn, v);
        }
    }
}

template <int LA, int LB, bool STORE, int AUX>
cudaError_t ris_launch_int_t(const RisGradParams& p, cudaStream_t st)
{
    const size_t smem = RIS_GRAD_WARPS * ris_int_warp_smem(p.pk.kmax, p.nb);
    if (smem > 48 * 1024) {          // per device and context: set at every launch that needs it, no process-wide cache
        const cudaError_t e = cudaFuncSetAttribute(ris_int_kernel<LA, LB, STORE, AUX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const int ny = (p.p1 - p.p0 + 31) / 32;
    const int nbt = (p.pk.ntasks + RIS_GRAD_WARPS - 1) / RIS_GRAD_WARPS;
    const int nx = std::max(1, std::min(nbt, (p.nsm * 3 + ny - 1) / ny));
    ris_int_kernel<LA, LB, STORE, AUX><<<dim3(nx, ny), RIS_GRAD_THREADS, smem, st>>>(p);
    return cudaGetLastError();
}

// p.aux_type: type of the auxiliary functions of the launch's list
template <int LA, int LB, bool STORE>
cudaError_t ris_launch_int(const RisGradParams& p, cudaStream_t st)
{
    if (p.pk.npairs <= 0 || p.pk.ntasks <= 0 || p.p1 <= p.p0) return cudaSuccess;
    if constexpr (STORE) {
        switch (p.aux_type) {
        case 0: return ris_launch_int_t<LA, LB, true, 0>(p, st);
        case 1: return ris_launch_int_t<LA, LB, true, 1>(p, st);
        case 2: return ris_launch_int_t<LA, LB, true, 2>(p, st);
        case 3: return ris_launch_int_t<LA, LB, true, 3>(p, st);
        default: return cudaErrorInvalidValue;
        }
    } else {
        switch (p.aux_type) {
        case 0: return ris_launch_int_t<LA, LB, false, 0>(p, st);
        case 1: return ris_launch_int_t<LA, LB, false, 1>(p, st);
        case 2: return ris_launch_int_t<LA, LB, false, 2>(p, st);
        case 3: return ris_launch_int_t<LA, LB, false, 3>(p, st);
        default: return cudaErrorInvalidValue;
        }
    }
}
