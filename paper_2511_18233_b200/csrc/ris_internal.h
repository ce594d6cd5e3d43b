// ris_internal.h -- structures shared between the translation units of libris_b200.so.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

constexpr int RIS_LMAX = 3;
constexpr int RIS_NCLASS = 10;          // (la,lb), la >= lb, la <= 3
constexpr int RIS_PRIM_FIELDS = 8;      // p, (P-Z)x, (P-Z)y, (P-Z)z, 1/(2p), 2a, 2b, coef   (Z = host centre)
constexpr int RIS_PAIR_PAD = 128;       // pairs per class padded to a multiple of this
constexpr int RIS_GRAD_THREADS = 128;

__host__ __device__ inline int ris_class_id(int la, int lb) { return la * (la + 1) / 2 + lb; }
__host__ __device__ inline int ris_ncart(int l) { return (l + 1) * (l + 2) / 2; }

// Packed shell pairs of one class (device pointers, SoA over the padded pair index).
struct RisClassPack {
    int la, lb;
    int npairs;            // surviving shell pairs
    int npad;              // padded count (multiple of RIS_PAIR_PAD); SoA stride
    int kmax;              // max surviving primitive pairs per shell pair
    long long nprim;       // surviving primitive pairs in the class
    double* geom;          // [6][npad]  Ax,Ay,Az, ABx,ABy,ABz  (AB = A - B)
    int* atoms;            // [2][npad]  atom of mu, atom of nu
    int* ao;               // [2][npad]  first AO of mu, first AO of nu
    int* nkA;              // [npad]     surviving primitive pairs hosted on A (a >= b); stored first
    int* nkB;              // [npad]     surviving primitive pairs hosted on B (b > a)
    float* symf;           // [npad]     1 (mu != nu shell) or 0.5 (same shell): folds D + D^T onto unique pairs
    double* prim;          // [kmax][8][npad]
    long long elem_off;    // offset of this class inside a packed tile slab
};

// Launch description of one class kernel (by value to the kernel).
struct RisGradParams {
    RisClassPack pk;
    int naux, natoms;
    const double* aux;       // [naux][5] Cx,Cy,Cz,alpha,auxfac
    const double* boys;      // table for M = E of this class
    const double* tile;      // packed tiles: + s*sstride + (P-p0)*pstride + elem_off + e*npad + ip
    long long sstride, pstride;
    const double* cscale;    // J: c_aux[nb][naux]; K: nullptr
    int nb;
    int p0, p1;              // aux range of this launch
    int pchunk;              // aux functions per blockIdx.y
    double* grad;            // [nb][natoms][3], accumulated with atomics
    unsigned long long* det; // deterministic mode: [nb][natoms][3][2] fixed-point accumulators (hi, lo), else nullptr
    int* det_flag;           // set to 1 when a contribution leaves the fixed-point range
};

// Deterministic reduction (ris_options.deterministic): a contribution x is added as the integer pair
//   hi = floor(x 2^28),  lo = floor((x 2^28 - hi) 2^32)        value = hi 2^-28 + lo 2^-60
// with two 64-bit INTEGER atomics; integer addition is associative, so the result does not depend on the order in
// which blocks arrive (resolution 2^-60 ~ 8.7e-19 per contribution, range |x| < 2^34, |sum| < 2^35).
__device__ __forceinline__ void ris_grad_add(const RisGradParams& prm, size_t idx, double x)
{
    if (prm.det == nullptr) { atomicAdd(prm.grad + idx, x); return; }
    if (!(fabs(x) < 17179869184.0)) { *prm.det_flag = 1; return; }
    const double y = x * 268435456.0;
    const long long hi = __double2ll_rd(y);
    const long long lo = __double2ll_rd((y - (double)hi) * 4294967296.0);
    atomicAdd(prm.det + 2 * idx, (unsigned long long)hi);
    atomicAdd(prm.det + 2 * idx + 1, (unsigned long long)lo);
}

typedef void (*ris_grad_launcher)(const RisGradParams&, cudaStream_t);
extern ris_grad_launcher ris_grad_launchers[RIS_NCLASS];
