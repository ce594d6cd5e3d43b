// ris_gemm.cuh -- S3-K1: the DGEMM-shaped Gamma^P assembly on the FP64 tensor path.
//   Gamma^P = C_occ B^P C_vir^T                     (AO back-transform, Eqs. 32-34, 39)
// evaluated as two "NT" contractions with K-contiguous operands:
//   GEMM-1   HT[nu'][(P,i)] = sum_a C_vir[nu][a] B[P][i][a]          nu' = spatial (Morton) position of AO nu
//   GEMM-2   S^P[mu'][nu']  = Gamma^P_{mu nu} + Gamma^P_{nu mu}
//                           = sum_i C_occ[mu][i] HT[nu'][(P,i)] + sum_i HT[mu'][(P,i)] C_occ[nu][i]
//            only for the 64x64 blocks of the spatially ordered AO index that contain a surviving shell pair
//            (block list), written as dense blocks that ris_k_pack_sym gathers into the packed pair order.
//
// One kernel serves both:  C[m][n] = sum_seg sum_k A_seg[row(m)][k] B_seg[n][k]  (up to two K segments; row(m)
// optionally through an index list, which is how GEMM-1 emits HT in spatial order).
// tcgen05.mma has no FP64 kind, so the tensor path for FP64 on sm_100a is the warp-level mma.sync f64 (DMMA;
// SASS DMMA.8x8x4); operands are staged global -> shared with cp.async (LDGSTS) in a 3-stage pipeline,
// fragments are read from shared memory with a row stride of 20 doubles (conflict-free for the 64-bit fragment
// pattern: row g, column t).
//   config A (GEMM-1): CTA tile 128x128, K step 16, 8 warps as 2 x 4, warp tile 64x32, 1 CTA/SM
//   config B (GEMM-2): CTA tile  64x64,  K step 16, 4 warps as 2 x 2, warp tile 32x32, 3 CTAs/SM
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

constexpr int RIS_GBK = 16, RIS_GLD = 20, RIS_GSTAGES = 3;
constexpr int RIS_GTILE2 = 64;           // AO block edge of the GEMM-2 block list

struct RisGemmSeg {
    const double* A; long long lda, bsA;   // A operand rows m, K contiguous; bsA = batch (blockIdx.z) stride in doubles
    const double* B; long long ldb, bsB;   // B operand rows n, K contiguous
    int K;
};

struct RisGemmParams {
    RisGemmSeg seg[2];
    int nseg;
    int M, N;
    const int* rowsA;                      // nullable: A row of output row m is rowsA[m] (segment 0 only)
    double* C; long long ldc, bsC;         // dense output: C[z*bsC + m*ldc + col(n)]
    int cdiv, cpad;                        // cdiv > 0: col(n) = (n / cdiv) * cpad + n % cdiv (padded sub-blocks); else col(n) = n
    const int2* tiles;                     // nullptr: grid.x = m-tile, grid.y = n-tile (dense).  Otherwise tile t =
    long long tile_stride;                 // blockIdx.x covers rows tiles[t].x*BM.., cols tiles[t].y*BN.. and is
                                           // written as a dense BM x BN block at C + z*bsC + t*tile_stride (ld BN)
};

template <bool VEC16>
__device__ __forceinline__ void ris_cp_async(unsigned smem, const double* gmem, int src_bytes)
{
    if (VEC16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem), "l"(gmem), "r"(src_bytes));
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(smem), "l"(gmem), "r"(src_bytes));
}

__device__ __forceinline__ void ris_dmma_16x8x8(double (&c)[4], const double (&a)[4], const double (&b)[2])
{
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+d"(c[0]), "+d"(c[1]), "+d"(c[2]), "+d"(c[3])
                 : "d"(a[0]), "d"(a[1]), "d"(a[2]), "d"(a[3]), "d"(b[0]), "d"(b[1]));
}

template <int BM, int BN, int WM, int WN>
struct RisGemmCfg {
    static constexpr int THREADS = (BM / WM) * (BN / WN) * 32;
    static constexpr int MT = WM / 16, NT = WN / 8;
    static constexpr size_t SMEM = (size_t)RIS_GSTAGES * (BM + BN) * RIS_GLD * sizeof(double);
};

// VEC16: all operand rows are 16-byte aligned (even leading dimensions, aligned bases) -> 16-byte cp.async
template <int BM, int BN, int WM, int WN, int MINB, bool VEC16>
__global__ void __launch_bounds__((BM / WM) * (BN / WN) * 32, MINB) ris_k_gemm_dmma(const RisGemmParams p)
{
    using Cfg = RisGemmCfg<BM, BN, WM, WN>;
    constexpr int THREADS = Cfg::THREADS, MT = Cfg::MT, NT = Cfg::NT;
    extern __shared__ __align__(16) double smem[];
    double* As = smem;                                          // [stage][BM][20]
    double* Bs = smem + (size_t)RIS_GSTAGES * BM * RIS_GLD;     // [stage][BN][20]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int wm0 = (warp / (BN / WN)) * WM, wn0 = (warp % (BN / WN)) * WN;
    int m0, n0;
    double* Cout;
    long long ldc;
    if (p.tiles) {
        const int2 tl = p.tiles[blockIdx.x];
        m0 = tl.x * BM; n0 = tl.y * BN;
        Cout = p.C + (long long)blockIdx.z * p.bsC + (long long)blockIdx.x * p.tile_stride;
        ldc = BN;
    } else {
        m0 = blockIdx.x * BM; n0 = blockIdx.y * BN;
        Cout = p.C + (long long)blockIdx.z * p.bsC + (long long)m0 * p.ldc + (p.cdiv > 0 ? 0 : n0);
        ldc = p.ldc;
    }
    const int nk0 = (p.seg[0].K + RIS_GBK - 1) / RIS_GBK;
    const int nk1 = p.nseg > 1 ? (p.seg[1].K + RIS_GBK - 1) / RIS_GBK : 0;
    const int nk = nk0 + nk1;

    // ---- loader state: one K step = BM (BN) rows x 16 doubles per operand; per-thread chunk pointers are
    // computed once per segment, the K loop only adds k0 and clamps the tail.
    constexpr int CH = VEC16 ? 8 : 16;                 // chunks per row
    constexpr int CW = VEC16 ? 2 : 1;                  // doubles per chunk
    constexpr int NA = BM * CH / THREADS, NB = BN * CH / THREADS;
    static_assert(BM * CH % THREADS == 0 && BN * CH % THREADS == 0, "loader mapping");
    const int kc = (tid % CH) * CW;
    const double* pa[NA];
    const double* pb[NB];
    int segK = 0;
    auto bind_segment = [&](int sidx) {
        const RisGemmSeg& sg = p.seg[sidx];
        segK = sg.K;
        const double* Ag = sg.A + (long long)blockIdx.z * sg.bsA;
        const double* Bg = sg.B + (long long)blockIdx.z * sg.bsB;
#pragma unroll
        for (int j = 0; j < NA; ++j) {
            const int r = m0 + (tid / CH) + j * (THREADS / CH);
            long long row = r;
            if (sidx == 0 && p.rowsA != nullptr && r < p.M) row = p.rowsA[r];
            pa[j] = r < p.M ? Ag + row * sg.lda + kc : nullptr;
        }
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            const int r = n0 + (tid / CH) + j * (THREADS / CH);
            pb[j] = r < p.N ? Bg + (long long)r * sg.ldb + kc : nullptr;
        }
    };
    const unsigned sA0 = (unsigned)__cvta_generic_to_shared(As) + ((tid / CH) * RIS_GLD + kc) * 8;
    const unsigned sB0 = (unsigned)__cvta_generic_to_shared(Bs) + ((tid / CH) * RIS_GLD + kc) * 8;
    int ld_ks = 0;                                     // next K step to load
    auto load_next = [&]() {
        if (ld_ks < nk) {
            if (ld_ks == 0) bind_segment(0);
            else if (ld_ks == nk0) bind_segment(1);
            const int k0 = (ld_ks < nk0 ? ld_ks : ld_ks - nk0) * RIS_GBK;
            const int stage = ld_ks % RIS_GSTAGES;
            const int kv = min(max(segK - (k0 + kc), 0), CW) * 8;               // valid bytes along K
#pragma unroll
            for (int j = 0; j < NA; ++j) {
                const bool v = pa[j] != nullptr && kv > 0;
                ris_cp_async<VEC16>(sA0 + (stage * BM + j * (THREADS / CH)) * RIS_GLD * 8, v ? pa[j] + k0 : p.seg[0].A, v ? kv : 0);
            }
#pragma unroll
            for (int j = 0; j < NB; ++j) {
                const bool v = pb[j] != nullptr && kv > 0;
                ris_cp_async<VEC16>(sB0 + (stage * BN + j * (THREADS / CH)) * RIS_GLD * 8, v ? pb[j] + k0 : p.seg[0].A, v ? kv : 0);
            }
        }
        ++ld_ks;
        asm volatile("cp.async.commit_group;");
    };

    double acc[MT][NT][4];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j)
#pragma unroll
            for (int r = 0; r < 4; ++r) acc[i][j][r] = 0.0;

#pragma unroll
    for (int s = 0; s < RIS_GSTAGES - 1; ++s) load_next();
    for (int ks = 0; ks < nk; ++ks) {
        asm volatile("cp.async.wait_group %0;" ::"n"(RIS_GSTAGES - 2));
        __syncthreads();
        load_next();                                   // refills the stage consumed in the previous iteration
        const double* as = As + (size_t)(ks % RIS_GSTAGES) * BM * RIS_GLD + (wm0 + g) * RIS_GLD + t;
        const double* bs = Bs + (size_t)(ks % RIS_GSTAGES) * BN * RIS_GLD + (wn0 + g) * RIS_GLD + t;
#pragma unroll
        for (int kk = 0; kk < RIS_GBK; kk += 8) {
            double a[MT][4], b[NT][2];
#pragma unroll
            for (int i = 0; i < MT; ++i) {
                a[i][0] = as[(16 * i) * RIS_GLD + kk];
                a[i][1] = as[(16 * i + 8) * RIS_GLD + kk];
                a[i][2] = as[(16 * i) * RIS_GLD + kk + 4];
                a[i][3] = as[(16 * i + 8) * RIS_GLD + kk + 4];
            }
#pragma unroll
            for (int j = 0; j < NT; ++j) {
                b[j][0] = bs[(8 * j) * RIS_GLD + kk];
                b[j][1] = bs[(8 * j) * RIS_GLD + kk + 4];
            }
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) ris_dmma_16x8x8(acc[i][j], a[i], b[j]);
        }
    }
    asm volatile("cp.async.wait_group 0;");

    // ---- epilogue: c0,c1 -> (row g, cols 2t, 2t+1); c2,c3 -> row g + 8
    const int Mrem = p.M - m0, Nrem = p.N - n0;
    const bool full = p.tiles != nullptr;              // block output: always a full BM x BN tile (zero padded)
    const bool vec = ((ldc & 1) == 0) && ((reinterpret_cast<uintptr_t>(Cout) & 15) == 0) && p.cdiv <= 0;
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int r = wm0 + 16 * i + g + 8 * h, c = wn0 + 8 * j + 2 * t;
                if (!full && r >= Mrem) continue;
                if (p.cdiv > 0) {                      // remapped columns (dense form only)
                    const int n = n0 + c;
                    if (c < Nrem) Cout[(long long)r * ldc + (long long)(n / p.cdiv) * p.cpad + n % p.cdiv] = acc[i][j][2 * h];
                    if (c + 1 < Nrem)
                        Cout[(long long)r * ldc + (long long)((n + 1) / p.cdiv) * p.cpad + (n + 1) % p.cdiv] = acc[i][j][2 * h + 1];
                    continue;
                }
                double* dst = Cout + (long long)r * ldc + c;
                if (vec && (full || c + 1 < Nrem)) {
                    *reinterpret_cast<double2*>(dst) = make_double2(acc[i][j][2 * h], acc[i][j][2 * h + 1]);
                } else {
                    if (full || c < Nrem) dst[0] = acc[i][j][2 * h];
                    if (full || c + 1 < Nrem) dst[1] = acc[i][j][2 * h + 1];
                }
            }
}

inline bool ris_gemm_aligned16(const RisGemmParams& p)
{
    for (int s = 0; s < p.nseg; ++s) {
        const RisGemmSeg& g = p.seg[s];
        if ((g.lda & 1) || (g.ldb & 1) || (g.bsA & 1) || (g.bsB & 1)) return false;
        if ((reinterpret_cast<uintptr_t>(g.A) & 15) || (reinterpret_cast<uintptr_t>(g.B) & 15)) return false;
    }
    return true;
}

template <int BM, int BN, int WM, int WN, int MINB>
inline cudaError_t ris_gemm_launch_cfg(cudaStream_t st, const RisGemmParams& p, int batch, int ntiles)
{
    using Cfg = RisGemmCfg<BM, BN, WM, WN>;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(ris_k_gemm_dmma<BM, BN, WM, WN, MINB, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(ris_k_gemm_dmma<BM, BN, WM, WN, MINB, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    dim3 grid;
    if (p.tiles) grid = dim3(ntiles, 1, batch);
    else grid = dim3((p.M + BM - 1) / BM, (p.N + BN - 1) / BN, batch);
    if (grid.x == 0 || grid.y == 0 || grid.z == 0) return cudaSuccess;
    if (ris_gemm_aligned16(p)) ris_k_gemm_dmma<BM, BN, WM, WN, MINB, true><<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(p);
    else ris_k_gemm_dmma<BM, BN, WM, WN, MINB, false><<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(p);
    return cudaGetLastError();
}

// GEMM-1: dense, 128x128 CTA tiles
inline cudaError_t ris_gemm_dense(cudaStream_t st, const RisGemmParams& p, int batch)
{
    return ris_gemm_launch_cfg<128, 128, 64, 32, 1>(st, p, batch, 0);
}
// GEMM-2: block list of RIS_GTILE2 x RIS_GTILE2 tiles
inline cudaError_t ris_gemm_blocks(cudaStream_t st, const RisGemmParams& p, int batch, int ntiles)
{
    return ris_gemm_launch_cfg<RIS_GTILE2, RIS_GTILE2, 32, 32, 3>(st, p, batch, ntiles);
}
