// ris_sph.cuh -- spherical-harmonic shells at the boundary (def2-TZVP is a spherical basis).
//
// With ris_options.spherical the caller's AO basis holds, per shell of degree l, the 2l+1 functions
//     chi_{lm}(r) = S_lm(r - A) sum_k d_k exp(-a_k |r - A|^2),   m = -l .. l  (in this order),
// S_lm = sqrt(4 pi/(2l+1)) r^l Y_lm^{real}: the real regular solid harmonics in Racah normalisation.  The integrals are linear
// in the bra functions, so the contractions over spherical functions are the Cartesian ones with
//     D_cart = U^T D_sph U,    C_cart = U^T C_sph       (U block diagonal, one (2l+1) x nc(l) block T_l per shell),
// and these two transforms are all that differs: the J tile packer folds U into its gather of D (no Cartesian D is ever
// stored), and the coefficient matrices of the K-type calls are expanded once per call.  Everything downstream (class kernels,
// GEMMs) runs on the Cartesian components it always had.
//
// T_l below is typed out polynomial by polynomial (Cartesian order lx descending, then ly descending):
//   l = 1:  y, z, x
//   l = 2:  sqrt3 xy, sqrt3 yz, zz - (xx + yy)/2, sqrt3 xz, (sqrt3/2)(xx - yy)
//   l = 3:  sqrt(5/8)(3 xxy - yyy), sqrt15 xyz, sqrt(3/8)(4 yzz - xxy - yyy), zzz - (3/2)(xxz + yyz),
//           sqrt(3/8)(4 xzz - xxx - xyy), (sqrt15/2)(xxz - yyz), sqrt(5/8)(xxx - 3 xyy)
#pragma once
#include "ris_internal.h"

#define RIS_S3 1.7320508075688772935      // sqrt(3)
#define RIS_S15 3.8729833462074168852     // sqrt(15)
#define RIS_S58 0.79056941504209483300    // sqrt(5/8)
#define RIS_S38 0.61237243569579452455    // sqrt(3/8)

// rows m = -l..l, columns the Cartesian components; offsets of the l blocks: 0, 1, 10, 40 (sizes 1, 9, 30, 70)
__device__ const double RIS_SPH_T[110] = {
    // l = 0
    1.0,
    // l = 1: x y z
    0.0, 1.0, 0.0,
    0.0, 0.0, 1.0,
    1.0, 0.0, 0.0,
    // l = 2: xx xy xz yy yz zz
    0.0, RIS_S3, 0.0, 0.0, 0.0, 0.0,
    0.0, 0.0, 0.0, 0.0, RIS_S3, 0.0,
    -0.5, 0.0, 0.0, -0.5, 0.0, 1.0,
    0.0, 0.0, RIS_S3, 0.0, 0.0, 0.0,
    0.5 * RIS_S3, 0.0, 0.0, -0.5 * RIS_S3, 0.0, 0.0,
    // l = 3: xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz
    0.0, 3.0 * RIS_S58, 0.0, 0.0, 0.0, 0.0, -RIS_S58, 0.0, 0.0, 0.0,
    0.0, 0.0, 0.0, 0.0, RIS_S15, 0.0, 0.0, 0.0, 0.0, 0.0,
    0.0, -RIS_S38, 0.0, 0.0, 0.0, 0.0, -RIS_S38, 0.0, 4.0 * RIS_S38, 0.0,
    0.0, 0.0, -1.5, 0.0, 0.0, 0.0, 0.0, -1.5, 0.0, 1.0,
    -RIS_S38, 0.0, 0.0, -RIS_S38, 0.0, 4.0 * RIS_S38, 0.0, 0.0, 0.0, 0.0,
    0.0, 0.0, 0.5 * RIS_S15, 0.0, 0.0, 0.0, 0.0, -0.5 * RIS_S15, 0.0, 0.0,
    RIS_S58, 0.0, 0.0, -3.0 * RIS_S58, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0,
};
__host__ __device__ constexpr int ris_sph_off(int l) { return l == 0 ? 0 : (l == 1 ? 1 : (l == 2 ? 10 : 40)); }

// J tiles from a density in the spherical basis (ris_k_pack_tiles): the tile element (ca, cb) of a pair is
//   sum_{m m'} T_la[m][ca] T_lb[m'][cb] (G[mu0 + m][nu0 + m'] + G[nu0 + m'][mu0 + m]),
// r0 / q0 = first spherical AO of the two shells, nao_s the spherical AO count.
__device__ __forceinline__ double ris_sph_pair_element(int la, int lb, int ca, int cb, size_t r0, size_t q0, int nao_s,
                                                       const double* __restrict__ g)
{
    const int nca = ris_ncart(la), ncb = ris_ncart(lb);
    const double* Ta = RIS_SPH_T + ris_sph_off(la) + ca;
    const double* Tb = RIS_SPH_T + ris_sph_off(lb) + cb;
    double v = 0.0;
    for (int m = 0; m < 2 * la + 1; ++m) {
        const double ta = Ta[m * nca];
        if (ta == 0.0) continue;
        double w = 0.0;
        for (int n = 0; n < 2 * lb + 1; ++n) {
            const double tb = Tb[n * ncb];
            if (tb != 0.0) w = fma(tb, g[(r0 + m) * nao_s + q0 + n] + g[(q0 + n) * nao_s + r0 + m], w);
        }
        v = fma(ta, w, v);
    }
    return v;
}

// Coefficient matrix to Cartesian rows: out[r][j] = sum_m T_l[m][comp(r)] C[sph0(r) + m][j], r over the Cartesian AOs;
// lc[r] = 16 l + component of r inside its shell.
__global__ void ris_k_sph_coef(int nao_c, int ncol, const int* __restrict__ sph0_of_ao, const int* __restrict__ lc,
                               const double* __restrict__ C, double* __restrict__ out)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)nao_c * ncol) return;
    const int r = (int)(idx / ncol), j = (int)(idx - (long long)r * ncol);
    const int l = lc[r] >> 4, comp = lc[r] & 15, nc = ris_ncart(l);
    const double* T = RIS_SPH_T + ris_sph_off(l) + comp;
    const double* src = C + (size_t)sph0_of_ao[r] * ncol + j;
    double v = 0.0;
    for (int m = 0; m < 2 * l + 1; ++m) {
        const double t = T[m * nc];
        if (t != 0.0) v = fma(t, src[(size_t)m * ncol], v);
    }
    out[idx] = v;
}
