// ris_gemm.cuh -- S3-K1: the DGEMM-shaped Gamma^P assembly on the FP64 tensor path.
//   Gamma^P = C_occ B^P C_vir^T                     (AO back-transform, Eqs. 32-34, 39)
// evaluated as two "NT" contractions with K-contiguous operands:
//   GEMM-1   HT[nu'][(P,i)] = sum_a C_vir[nu][a] B[P][i][a]          nu' = spatial (Morton) position of AO nu
//   GEMM-2   X^P[mu'][nu']  = Gamma^P_{mu nu} = sum_i C_occ[mu][i] HT[nu'][(P,i)]   for the SURVIVING (mu, nu) only,
//            one problem per AO column nu' with P as the dense N dimension:
//                X_nu'[m][P] = sum_i C_occ[partner_m(nu')][i] HT[nu'][(P,i)],
//            m over the GATHERED list of nu's surviving partners (no tile cover of a sparse matrix: the only padding
//            is the tail of a partner list and of the P range), and the result is ADDED (red.global.add.f64), times
//            the pair's symmetry factor, straight into the P-minor packed K tile of the class kernels:
//                tile[element(mu,nu)][P] += f X^P[mu'][nu'];   every element receives exactly its two halves
//            Gamma^P_{mu nu} and Gamma^P_{nu mu} (one for a diagonal element), so the sum is order-independent.
//            (Round 1 computed S^P = Gamma^P + Gamma^P^T on 32 x 64 tiles covering the sparse pair matrix -- 1.7x the
//            algorithmic flops -- into a block buffer that a second kernel transposed into the tiles.)
//
// One kernel serves both:  C[m][n] = sum_seg sum_k A_seg[row(m)][k] B_seg[n][k]  (up to two K segments; row(m)
// optionally through an index list, which is how GEMM-1 emits HT in spatial order and GEMM-2 gathers its partners).
// tcgen05.mma has no FP64 kind, so the tensor path for FP64 on sm_100a is the warp-level mma.sync f64 (DMMA;
// SASS DMMA.8x8x4, 16 cycles of the pipe per SM sub-partition each).  Operands are staged global -> shared with
// cp.async (LDGSTS) through a multi-stage pipeline that is synchronised by mbarriers only (full[s]: the stage's
// cp.async have landed; empty[s]: every warp has read its fragments) -- a CTA-wide barrier per K step cost 15 % of the
// DMMA pipe (measured in round 1).  Fragments are read with 128-bit shared loads from a
// 16-double row whose halves are swapped on odd rows (bank-conflict free, no padding).
//   GEMM-1: CTA tile 64x128, K step 16, 8 warps as 2 x 4, warp tile 32x32, 3 stages, 2 CTAs/SM
//   GEMM-2: CTA tile 64x64 (partners x aux),  K step 16, 4 warps as 2 x 2, warp tile 32x32, 3 stages, 3 CTAs/SM
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

constexpr int RIS_GBK = 16, RIS_GLD = 16;   // K step; shared row stride in doubles (swizzled, see the kernel)
constexpr int RIS_GTILE2 = 64;           // AO block edge of the fit_K bands (spatial AO order)

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
    int cdiv; long long cpad;              // cdiv > 0: col(n) = (n / cdiv) * cpad + n % cdiv (padded sub-blocks); else col(n) = n
    const int2* tiles;                     // nullptr: grid.x = m-tile, grid.y = n-tile (dense).  Otherwise tile t =
    long long tile_stride;                 // blockIdx.x covers rows tiles[t].x*BM.., cols tiles[t].y*BN.. and is
                                           // written as a dense BM x BN block at C + z*bsC + t*tile_stride (ld BN)
    const int* gcols;                      // nullable, with tiles: GATHERED columns -- column n of tile t is the B row
                                           // gcols[tiles[t].y + n] (< 0: padding, zero column); tiles[t].y is then an
                                           // offset into gcols, not a block index
    // SCATTER mode (template SCAT; GEMM-2): tile t = blockIdx.x is (column problem nu = tiles[t].x, first entry m0 =
    // tiles[t].y of its partner list); row m of the tile is A row srows[m0 + m] (< 0: padding); B of problem nu starts
    // at seg[0].B + nu * seg[0].bsB; blockIdx.y = n-tile; the result row m is ADDED to
    // C[(scode[m0 + m] >> 1) * ldc + n] times (scode & 1 ? 0.5 : 1).
    const int* srows;
    const int* scode;
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

template <int BM, int BN, int WM, int WN, int STAGES>
struct RisGemmCfg {
    static constexpr int THREADS = (BM / WM) * (BN / WN) * 32;
    static constexpr int MT = WM / 16, NT = WN / 8;
    static constexpr size_t SMEM = (size_t)STAGES * (BM + BN) * RIS_GLD * sizeof(double);
};

// VEC16: all operand rows are 16-byte aligned (even leading dimensions, aligned bases) -> 16-byte cp.async
// GATH: gathered-column tiles (p.gcols); a warp whose WN-column strip is all padding issues no MMAs (skipping single
// 8-column sub-tiles was measured slower: the predicates break the MMA schedule, 48.2 -> 49.8 ms on config 4).
template <int BM, int BN, int WM, int WN, int STAGES, int MINB, bool VEC16, bool GATH = false, bool SCAT = false>
__global__ void __launch_bounds__((BM / WM) * (BN / WN) * 32, MINB) ris_k_gemm_dmma(const RisGemmParams p)
{
    using Cfg = RisGemmCfg<BM, BN, WM, WN, STAGES>;
    constexpr int THREADS = Cfg::THREADS, MT = Cfg::MT, NT = Cfg::NT;
    extern __shared__ __align__(16) double smem[];
    double* As = smem;                                     // [stage][BM][16]
    double* Bs = smem + (size_t)STAGES * BM * RIS_GLD;     // [stage][BN][16]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int wm0 = (warp / (BN / WN)) * WM, wn0 = (warp % (BN / WN)) * WN;
    int m0, n0;
    double* Cout;
    long long ldc;
    int snu = 0;                                       // SCAT: the column problem of this tile
    if (SCAT) {
        const int2 tl = p.tiles[blockIdx.x];
        snu = tl.x; m0 = tl.y; n0 = blockIdx.y * BN;
        Cout = p.C; ldc = p.ldc;
    } else if (p.tiles) {
        const int2 tl = p.tiles[blockIdx.x];
        m0 = tl.x * BM; n0 = p.gcols ? tl.y : tl.y * BN;
        Cout = p.C + (long long)blockIdx.z * p.bsC + (long long)blockIdx.x * p.tile_stride;
        ldc = BN;
    } else {
        m0 = blockIdx.x * BM; n0 = blockIdx.y * BN;
        Cout = p.C + (long long)blockIdx.z * p.bsC + (long long)m0 * p.ldc + (p.cdiv > 0 ? 0 : n0);
        ldc = p.ldc;
    }
    int nvw = WN;                                      // valid (non-padding) columns of this warp's WN-column strip
    if (GATH) {
        int cnt = 0;
        for (int c0 = lane; c0 < WN; c0 += 32) cnt += p.gcols[n0 + wn0 + c0] >= 0 ? 1 : 0;
        for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
        nvw = cnt;                                     // padding sits at the end of a panel's list only
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
        const double* Bg = sg.B + (long long)(SCAT ? snu : blockIdx.z) * sg.bsB;
#pragma unroll
        for (int j = 0; j < NA; ++j) {
            const int r = m0 + (tid / CH) + j * (THREADS / CH);
            if (SCAT) {
                const int row = p.srows[r];            // the partner lists are padded to whole tiles
                pa[j] = row >= 0 ? Ag + (long long)row * sg.lda + kc : nullptr;
                continue;
            }
            long long row = r;
            if (sidx == 0 && p.rowsA != nullptr && r < p.M) row = p.rowsA[r];
            pa[j] = r < p.M ? Ag + row * sg.lda + kc : nullptr;
        }
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            int r = n0 + (tid / CH) + j * (THREADS / CH);
            if (p.gcols != nullptr) r = p.gcols[r];          // gathered column: B row index, or -1 (padding)
            pb[j] = (r >= 0 && r < p.N) ? Bg + (long long)r * sg.ldb + kc : nullptr;
        }
    };
    // shared layout: row stride RIS_GLD = 16 doubles (one K step), the two 8-double halves of odd rows swapped
    // (k' = k ^ 8 (row & 1)): the 8 lanes of a quarter warp (rows g, g+1; t = 0..3) of a 128-bit fragment load then
    // cover all 32 banks once, without padding.
    const int lrow = tid / CH;                         // loader row (same parity for every j: THREADS / CH is even)
    const int lk = kc ^ ((lrow & 1) << 3);
    const unsigned sA0 = (unsigned)__cvta_generic_to_shared(As) + (lrow * RIS_GLD + lk) * 8;
    const unsigned sB0 = (unsigned)__cvta_generic_to_shared(Bs) + (lrow * RIS_GLD + lk) * 8;
    // ---- pipeline: STAGES shared stages, no CTA-wide barrier in the K loop.  full[s] completes when every thread's
    // cp.async of the stage has landed (cp.async.mbarrier.arrive.noinc, count THREADS); empty[s] when every warp has
    // read its fragments (count NWARPS).  K step j is issued DIST = STAGES - 2 steps ahead, into the stage all warps
    // left two steps ago, so warps drift apart by up to a step instead of meeting at a barrier.
    constexpr int NWARPS = THREADS / 32, DIST = STAGES - 2;
    static_assert(STAGES >= 3, "pipeline depth");
    __shared__ __align__(8) unsigned long long bars[2 * STAGES];
    const unsigned bar0 = (unsigned)__cvta_generic_to_shared(bars);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar0 + 8 * s), "r"(THREADS));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar0 + 8 * (STAGES + s)), "r"(NWARPS));
        }
    }
    __syncthreads();
    auto bar_wait = [&](unsigned bar, int parity) {
        unsigned done;
        do {
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                         : "=r"(done) : "r"(bar), "r"(parity) : "memory");
        } while (!done);
    };
    auto produce = [&](int j) {
        if (j >= nk) return;
        if (j == 0) bind_segment(0);
        else if (j == nk0) bind_segment(1);
        const int k0 = (j < nk0 ? j : j - nk0) * RIS_GBK;
        const int stage = j % STAGES, round = j / STAGES;
        if (round > 0) bar_wait(bar0 + 8 * (STAGES + stage), (round - 1) & 1);
        const int kv = min(max(segK - (k0 + kc), 0), CW) * 8;               // valid bytes along K
#pragma unroll
        for (int jj = 0; jj < NA; ++jj) {
            const bool v = pa[jj] != nullptr && kv > 0;
            ris_cp_async<VEC16>(sA0 + (stage * BM + jj * (THREADS / CH)) * RIS_GLD * 8, v ? pa[jj] + k0 : p.seg[0].A, v ? kv : 0);
        }
#pragma unroll
        for (int jj = 0; jj < NB; ++jj) {
            const bool v = pb[jj] != nullptr && kv > 0;
            ris_cp_async<VEC16>(sB0 + (stage * BN + jj * (THREADS / CH)) * RIS_GLD * 8, v ? pb[jj] + k0 : p.seg[0].A, v ? kv : 0);
        }
        asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar0 + 8 * stage) : "memory");
    };

    double acc[MT][NT][4];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j)
#pragma unroll
            for (int r = 0; r < 4; ++r) acc[i][j][r] = 0.0;

#pragma unroll
    for (int j = 0; j < DIST; ++j) produce(j);
    const int ksw = (g & 1) << 3;
    for (int ks = 0; ks < nk; ++ks) {
        produce(ks + DIST);
        const int stage = ks % STAGES;
        bar_wait(bar0 + 8 * stage, (ks / STAGES) & 1);
        // Fragments, K-permuted: the MMA's k index t (t + 4) is the shared column kk + 2t (kk + 2t + 1) for A and B
        // alike, so one 128-bit load fetches both k halves of a fragment row.
        const double* as = As + (size_t)stage * BM * RIS_GLD + (wm0 + g) * RIS_GLD + 2 * t;
        const double* bs = Bs + (size_t)stage * BN * RIS_GLD + (wn0 + g) * RIS_GLD + 2 * t;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            double a[MT][4], b[NT][2];
            const int kk = (8 * h) ^ ksw;
#pragma unroll
            for (int i = 0; i < MT; ++i) {
                const double2 lo = *reinterpret_cast<const double2*>(as + (16 * i) * RIS_GLD + kk);
                const double2 hi = *reinterpret_cast<const double2*>(as + (16 * i + 8) * RIS_GLD + kk);
                a[i][0] = lo.x; a[i][1] = hi.x; a[i][2] = lo.y; a[i][3] = hi.y;
            }
#pragma unroll
            for (int j = 0; j < NT; ++j) {
                const double2 v = *reinterpret_cast<const double2*>(bs + (8 * j) * RIS_GLD + kk);
                b[j][0] = v.x; b[j][1] = v.y;
            }
            if (h == 1) {          // every fragment of the stage is in registers: release it before the last MMAs
                __syncwarp();
                if (lane == 0) {
                    unsigned long long st_;
                    asm volatile("mbarrier.arrive.shared::cta.b64 %0, [%1];" : "=l"(st_) : "r"(bar0 + 8 * (STAGES + stage)) : "memory");
                }
            }
            if (GATH && nvw == 0) continue;            // warp-uniform: the whole strip is padding
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) ris_dmma_16x8x8(acc[i][j], a[i], b[j]);
        }
    }

    // ---- epilogue: c0,c1 -> (row g, cols 2t, 2t+1); c2,c3 -> row g + 8
    if (SCAT) {
        const int Nr = p.N - n0;
#pragma unroll
        for (int i = 0; i < MT; ++i)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int code = p.scode[m0 + wm0 + 16 * i + g + 8 * h];
                if (code < 0) continue;
                const double f = (code & 1) ? 0.5 : 1.0;
                double* dst = Cout + (long long)(code >> 1) * ldc + n0;
#pragma unroll
                for (int j = 0; j < NT; ++j) {
                    const int c = wn0 + 8 * j + 2 * t;
                    // (PTX has no vector form of red.add.f64: two 8-byte reductions into one 16-byte piece of the row)
                    if (c < Nr) atomicAdd(dst + c, f * acc[i][j][2 * h]);
                    if (c + 1 < Nr) atomicAdd(dst + c + 1, f * acc[i][j][2 * h + 1]);
                }
            }
        return;
    }
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

template <int BM, int BN, int WM, int WN, int STAGES, int MINB, bool GATH = false, bool SCAT = false>
inline cudaError_t ris_gemm_launch_cfg(cudaStream_t st, const RisGemmParams& p, int batch, int ntiles)
{
    using Cfg = RisGemmCfg<BM, BN, WM, WN, STAGES>;
    const bool vec16 = ris_gemm_aligned16(p);
    if (Cfg::SMEM + 1024 > 48 * 1024) {     // (+ the static barriers) per device and context: set at every launch that needs
                                            // it, no process-wide cache
        const cudaError_t e = vec16 ? cudaFuncSetAttribute(ris_k_gemm_dmma<BM, BN, WM, WN, STAGES, MINB, true, GATH, SCAT>,
                                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM)
                                    : cudaFuncSetAttribute(ris_k_gemm_dmma<BM, BN, WM, WN, STAGES, MINB, false, GATH, SCAT>,
                                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
        if (e != cudaSuccess) return e;
    }
    dim3 grid;
    if (SCAT) grid = dim3(ntiles, (p.N + BN - 1) / BN, 1);
    else if (p.tiles) grid = dim3(ntiles, 1, batch);
    else grid = dim3((p.M + BM - 1) / BM, (p.N + BN - 1) / BN, batch);
    if (grid.x == 0 || grid.y == 0 || grid.z == 0) return cudaSuccess;
    if (vec16) ris_k_gemm_dmma<BM, BN, WM, WN, STAGES, MINB, true, GATH, SCAT><<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(p);
    else ris_k_gemm_dmma<BM, BN, WM, WN, STAGES, MINB, false, GATH, SCAT><<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(p);
    return cudaGetLastError();
}

// GEMM-1: dense, CTA tile 64x128, 8 warps (2 x 4, warp tile 32x32), 3 stages, 2 CTAs/SM.  Measured on B200 (config 4,
// round 1; now profiles/r02_v1_ncu.md): 33.2 TFLOP/s = 90 % of the mma.sync f64 peak; 128x128 tiles with 8 or 16 warps on one
// CTA/SM reach 31.3-31.6, 128x64 x 2 CTAs 31.9, the same tile with 4 stages 32.4.
inline cudaError_t ris_gemm_dense(cudaStream_t st, const RisGemmParams& p, int batch)
{
#ifndef RIS_G1_STAGES
#define RIS_G1_STAGES 3
#endif
    return ris_gemm_launch_cfg<64, 128, 32, 32, RIS_G1_STAGES, 2>(st, p, batch, 0);
}
// GEMM-2 (scatter mode): tiles of RIS_G2_BM gathered partner rows x RIS_G2_BN aux functions, K = nocc
#ifndef RIS_G2_BM
#define RIS_G2_BM 64            // measured on config 4 (r02): 64x64 / 3 CTAs 29.8 ms per step, 32x64 / 5 CTAs 30.2, / 6 CTAs
                                // (skipping the MMAs of a warp whose 32-row strip is all padding: 30.9 -- left out)
#define RIS_G2_BN 64            // 30.3, 32x64 with 4 stages 32.5
#define RIS_G2_STAGES 3
#define RIS_G2_MINB 3
#endif
inline cudaError_t ris_gemm_scatter(cudaStream_t st, const RisGemmParams& p, int ntiles)
{
    // up to 32 auxiliary functions (molecules of a few tens of atoms): one 32-column tile, 2 warps per CTA -- half the padded
    // MMA work and shared memory of the 64-column tile
    if (p.N <= 32) return ris_gemm_launch_cfg<RIS_G2_BM, 32, 32, 32, RIS_G2_STAGES, 6, false, true>(st, p, 1, ntiles);
    // the aux index is the N dimension and is padded to whole tiles: take the tile width (64, 96 or 112 columns; 2 x 2 warps
    // of 32 x 32 / 48 / 56) that pads least -- 100 functions: 112 instead of 128, 84: 96, 300: 320 (ties: the 64-column tile)
    const int pad64 = (p.N + 63) / 64 * 64, pad96 = (p.N + 95) / 96 * 96, pad112 = (p.N + 111) / 112 * 112;
    if (pad112 < pad64 && pad112 <= pad96)
        return ris_gemm_launch_cfg<RIS_G2_BM, 112, 32, 56, RIS_G2_STAGES, RIS_G2_MINB, false, true>(st, p, 1, ntiles);
    if (pad96 < pad64)
        return ris_gemm_launch_cfg<RIS_G2_BM, 96, 32, 48, RIS_G2_STAGES, RIS_G2_MINB, false, true>(st, p, 1, ntiles);
    return ris_gemm_launch_cfg<RIS_G2_BM, RIS_G2_BN, 32, 32, RIS_G2_STAGES, RIS_G2_MINB, false, true>(st, p, 1, ntiles);
}
