// ris_gemm.cuh -- S3-K1: the DGEMM-shaped Gamma^P assembly
//   H^P = B^P C_vir^T,  Gamma^P = C_occ H^P      (Gamma = C_occ B C_vir^T: Eqs. 32-34, 39)
// Batched row-major FP64 GEMM, C[z] = A[z] * op(B[z]):
//   BT = true :  C[M][N] = A[M][K] * B[N][K]^T
//   BT = false:  C[M][N] = A[M][K] * B[K][N]
// v1: 64x64x16 shared-memory tiles, 256 threads, 4x4 register micro-tile on the FP64 FMA pipe.
#pragma once
#include <cuda_runtime.h>

constexpr int RIS_GM = 64, RIS_GN = 64, RIS_GK = 16;

template <bool BT>
__global__ void __launch_bounds__(256) ris_k_gemm(int M, int N, int K, const double* __restrict__ A, int lda, long long sA,
                                                  const double* __restrict__ B, int ldb, long long sB,
                                                  double* __restrict__ C, int ldc, long long sC)
{
    __shared__ double As[RIS_GK][RIS_GM + 4];
    __shared__ double Bs[RIS_GK][RIS_GN + 4];
    A += (size_t)blockIdx.z * sA; B += (size_t)blockIdx.z * sB; C += (size_t)blockIdx.z * sC;
    const int m0 = blockIdx.y * RIS_GM, n0 = blockIdx.x * RIS_GN;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    double acc[4][4] = {};
    for (int k0 = 0; k0 < K; k0 += RIS_GK) {
        // A tile: 64 rows x 16 k (k contiguous in memory)
        for (int i = threadIdx.x; i < RIS_GM * RIS_GK; i += 256) {
            const int r = i / RIS_GK, kk = i % RIS_GK;
            const int gm = m0 + r, gk = k0 + kk;
            As[kk][r] = (gm < M && gk < K) ? A[(size_t)gm * lda + gk] : 0.0;
        }
        if (BT) {
            for (int i = threadIdx.x; i < RIS_GN * RIS_GK; i += 256) {
                const int r = i / RIS_GK, kk = i % RIS_GK;
                const int gn = n0 + r, gk = k0 + kk;
                Bs[kk][r] = (gn < N && gk < K) ? B[(size_t)gn * ldb + gk] : 0.0;
            }
        } else {
            for (int i = threadIdx.x; i < RIS_GN * RIS_GK; i += 256) {
                const int kk = i / RIS_GN, r = i % RIS_GN;
                const int gn = n0 + r, gk = k0 + kk;
                Bs[kk][r] = (gn < N && gk < K) ? B[(size_t)gk * ldb + gn] : 0.0;
            }
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < RIS_GK; ++kk) {
            double a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) { a[i] = As[kk][ty * 4 + i]; b[i] = Bs[kk][tx * 4 + i]; }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int gm = m0 + ty * 4 + i, gn = n0 + tx * 4 + j;
            if (gm < M && gn < N) C[(size_t)gm * ldc + gn] = acc[i][j];
        }
}

template <bool BT>
inline void ris_gemm(cudaStream_t st, int M, int N, int K, const double* A, int lda, long long sA, const double* B, int ldb,
                     long long sB, double* C, int ldc, long long sC, int batch)
{
    dim3 grid((N + RIS_GN - 1) / RIS_GN, (M + RIS_GM - 1) / RIS_GM, batch);
    ris_k_gemm<BT><<<grid, 256, 0, st>>>(M, N, K, A, lda, sA, B, ldb, sB, C, ldc, sC);
}
