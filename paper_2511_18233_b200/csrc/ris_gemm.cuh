// ris_gemm.cuh -- S3-K1: the DGEMM-shaped Gamma^P assembly on the FP64 tensor path.
//   Gamma^P = C_occ B^P C_vir^T                     (AO back-transform, Eqs. 32-34, 39)
// evaluated as two "NT" contractions with K-contiguous operands:
//   GEMM-1   HT[nu][(P,i)]  = sum_a C_vir[nu][a] B[P][i][a]
//   GEMM-2   S^P[mu][nu]    = Gamma^P_{mu nu} + Gamma^P_{nu mu}
//                           = sum_i C_occ[mu][i] HT[nu][(P,i)] + sum_i HT[mu][(P,i)] C_occ[nu][i]
//            only for the 128x128 AO blocks that contain a surviving shell pair (block list), written as
//            dense blocks that ris_k_pack_sym gathers into the packed pair order.
//
// One kernel serves both:  C[m][n] = sum_seg sum_k A_seg[m][k] B_seg[n][k]  (up to two K segments).
// tcgen05.mma has no FP64 kind, so the tensor path for FP64 on sm_100a is the warp-level
// mma.sync.m16n8k8.f64 (DMMA); operands are staged global -> shared with cp.async (LDGSTS) in a
// 3-stage pipeline, fragments are read from shared memory with a row stride of 20 doubles (conflict-free
// for the 64-bit fragment pattern: row g, column t).
//   CTA tile 128x128, K step 16, 8 warps as 2 (M) x 4 (N), warp tile 64x32 = 4 x 4 MMA tiles, 64 FP64
//   accumulators per thread.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

constexpr int RIS_GBM = 128, RIS_GBN = 128, RIS_GBK = 16, RIS_GLD = 20, RIS_GSTAGES = 3, RIS_GTHREADS = 256;
constexpr size_t RIS_GEMM_SMEM = (size_t)RIS_GSTAGES * (RIS_GBM + RIS_GBN) * RIS_GLD * sizeof(double);

struct RisGemmSeg {
    const double* A; long long lda, bsA;   // A operand rows m, K contiguous; bsA = batch (blockIdx.z) stride in doubles
    const double* B; long long ldb, bsB;   // B operand rows n, K contiguous
    int K;
};

struct RisGemmParams {
    RisGemmSeg seg[2];
    int nseg;
    int M, N;
    double* C; long long ldc, bsC;         // dense output: C[z*bsC + m*ldc + col(n)]
    int cdiv, cpad;                        // cdiv > 0: col(n) = (n / cdiv) * cpad + n % cdiv (padded sub-blocks); else col(n) = n
    const int2* tiles;                     // nullptr: grid.x = m-tile, grid.y = n-tile (dense).  Otherwise tile t =
    long long tile_stride;                 // blockIdx.x covers rows tiles[t].x*128.., cols tiles[t].y*128.. and is
                                           // written as a dense 128x128 block at C + z*bsC + t*tile_stride (ld 128)
};

__device__ __forceinline__ void ris_cp_async(double* smem, const double* gmem, int src_bytes, bool vec16)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    if (vec16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(src_bytes));
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(s), "l"(gmem), "r"(src_bytes));
}

__device__ __forceinline__ void ris_dmma_16x8x8(double (&c)[4], const double (&a)[4], const double (&b)[2])
{
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+d"(c[0]), "+d"(c[1]), "+d"(c[2]), "+d"(c[3])
                 : "d"(a[0]), "d"(a[1]), "d"(a[2]), "d"(a[3]), "d"(b[0]), "d"(b[1]));
}

// VEC16: all operand rows are 16-byte aligned (even leading dimensions, aligned bases) -> 16-byte cp.async
template <bool VEC16>
__global__ void __launch_bounds__(RIS_GTHREADS, 1) ris_k_gemm_dmma(const RisGemmParams p)
{
    extern __shared__ __align__(16) double smem[];
    double* As = smem;                                              // [stage][128][20]
    double* Bs = smem + (size_t)RIS_GSTAGES * RIS_GBM * RIS_GLD;    // [stage][128][20]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int wm0 = (warp >> 2) * 64, wn0 = (warp & 3) * 32;
    int m0, n0;
    double* Cout;
    long long ldc;
    if (p.tiles) {
        const int2 tl = p.tiles[blockIdx.x];
        m0 = tl.x * RIS_GBM; n0 = tl.y * RIS_GBN;
        Cout = p.C + (long long)blockIdx.z * p.bsC + (long long)blockIdx.x * p.tile_stride;
        ldc = RIS_GBN;
    } else {
        m0 = blockIdx.x * RIS_GBM; n0 = blockIdx.y * RIS_GBN;
        Cout = p.C + (long long)blockIdx.z * p.bsC + (long long)m0 * p.ldc + (p.cdiv > 0 ? 0 : n0);
        ldc = p.ldc;
    }
    const int nk0 = (p.seg[0].K + RIS_GBK - 1) / RIS_GBK;
    const int nk1 = p.nseg > 1 ? (p.seg[1].K + RIS_GBK - 1) / RIS_GBK : 0;
    const int nk = nk0 + nk1;

    // loader: one K step = 128 rows x 16 doubles per operand
    constexpr int CH = VEC16 ? 8 : 16;                 // chunks per row
    constexpr int CW = VEC16 ? 2 : 1;                  // doubles per chunk
    constexpr int PER_THREAD = RIS_GBM * CH / RIS_GTHREADS;
    auto load_stage = [&](int ks, int stage) {
        const RisGemmSeg& sg = ks < nk0 ? p.seg[0] : p.seg[1];
        const int k0 = (ks < nk0 ? ks : ks - nk0) * RIS_GBK;
        const double* Ag = sg.A + (long long)blockIdx.z * sg.bsA;
        const double* Bg = sg.B + (long long)blockIdx.z * sg.bsB;
        double* as = As + (size_t)stage * RIS_GBM * RIS_GLD;
        double* bs = Bs + (size_t)stage * RIS_GBN * RIS_GLD;
#pragma unroll
        for (int j = 0; j < PER_THREAD; ++j) {
            const int c = tid + j * RIS_GTHREADS;
            const int r = c / CH, kc = (c % CH) * CW;
            const int kv = min(max(sg.K - (k0 + kc), 0), CW) * 8;             // valid bytes along K
            const int ra = m0 + r, rb = n0 + r;
            const bool va = ra < p.M && kv > 0, vb = rb < p.N && kv > 0;
            ris_cp_async(as + r * RIS_GLD + kc, va ? Ag + (long long)ra * sg.lda + k0 + kc : Ag, va ? kv : 0, VEC16);
            ris_cp_async(bs + r * RIS_GLD + kc, vb ? Bg + (long long)rb * sg.ldb + k0 + kc : Bg, vb ? kv : 0, VEC16);
        }
    };

    double acc[4][4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int r = 0; r < 4; ++r) acc[i][j][r] = 0.0;

#pragma unroll
    for (int s = 0; s < RIS_GSTAGES - 1; ++s) {
        if (s < nk) load_stage(s, s);
        asm volatile("cp.async.commit_group;");
    }
    for (int ks = 0; ks < nk; ++ks) {
        asm volatile("cp.async.wait_group %0;" ::"n"(RIS_GSTAGES - 2));
        __syncthreads();
        {   // prefetch the stage that was consumed in the previous iteration
            const int nx = ks + RIS_GSTAGES - 1;
            if (nx < nk) load_stage(nx, nx % RIS_GSTAGES);
            asm volatile("cp.async.commit_group;");
        }
        const double* as = As + (size_t)(ks % RIS_GSTAGES) * RIS_GBM * RIS_GLD + (wm0 + g) * RIS_GLD + t;
        const double* bs = Bs + (size_t)(ks % RIS_GSTAGES) * RIS_GBN * RIS_GLD + (wn0 + g) * RIS_GLD + t;
#pragma unroll
        for (int kk = 0; kk < RIS_GBK; kk += 8) {
            double a[4][4], b[4][2];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                a[i][0] = as[(16 * i) * RIS_GLD + kk];
                a[i][1] = as[(16 * i + 8) * RIS_GLD + kk];
                a[i][2] = as[(16 * i) * RIS_GLD + kk + 4];
                a[i][3] = as[(16 * i + 8) * RIS_GLD + kk + 4];
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                b[j][0] = bs[(8 * j) * RIS_GLD + kk];
                b[j][1] = bs[(8 * j) * RIS_GLD + kk + 4];
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) ris_dmma_16x8x8(acc[i][j], a[i], b[j]);
        }
    }
    asm volatile("cp.async.wait_group 0;");

    // epilogue: c0,c1 -> (row g, cols 2t, 2t+1); c2,c3 -> row g + 8
    const int Mrem = p.M - m0, Nrem = p.N - n0;
    const bool vec = ((ldc & 1) == 0) && ((reinterpret_cast<uintptr_t>(Cout) & 15) == 0) && p.cdiv <= 0;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int r = wm0 + 16 * i + g + 8 * h, c = wn0 + 8 * j + 2 * t;
                const bool full = p.tiles != nullptr;          // block output: always a full 128x128 tile (zero padded)
                if (!full && r >= Mrem) continue;
                double* dst = Cout + (long long)r * ldc + c;
                if (p.cdiv > 0) {          // remapped columns (dense form only)
                    const int n = n0 + c;
                    if (c < Nrem) Cout[(long long)r * ldc + (long long)(n / p.cdiv) * p.cpad + n % p.cdiv] = acc[i][j][2 * h];
                    if (c + 1 < Nrem) Cout[(long long)r * ldc + (long long)((n + 1) / p.cdiv) * p.cpad + (n + 1) % p.cdiv] = acc[i][j][2 * h + 1];
                    continue;
                }
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

// batch = gridDim.z; ntiles > 0 selects the block-list form
inline cudaError_t ris_gemm_launch(cudaStream_t st, const RisGemmParams& p, int batch, int ntiles)
{
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(ris_k_gemm_dmma<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RIS_GEMM_SMEM);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(ris_k_gemm_dmma<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RIS_GEMM_SMEM);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    dim3 grid;
    if (p.tiles) grid = dim3(ntiles, 1, batch);
    else grid = dim3((p.M + RIS_GBM - 1) / RIS_GBM, (p.N + RIS_GBN - 1) / RIS_GBN, batch);
    if (grid.x == 0 || grid.y == 0 || grid.z == 0) return cudaSuccess;
    if (ris_gemm_aligned16(p)) ris_k_gemm_dmma<true><<<grid, RIS_GTHREADS, RIS_GEMM_SMEM, st>>>(p);
    else ris_k_gemm_dmma<false><<<grid, RIS_GTHREADS, RIS_GEMM_SMEM, st>>>(p);
    return cudaGetLastError();
}
