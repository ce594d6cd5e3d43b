// ris_setup.cuh -- S0: shell-pair screening, sorting by (l_mu,l_nu) class and SoA
// packing, all on the device.  The paper is silent on screening / ordering; the bound
// is the one documented in include/ris.h (ris_options.schwarz_tol).
#pragma once
#include "ris_internal.h"

struct RisMolDev {
    int natoms, nshells;
    const double* coords;
    const int *shell_atom, *shell_l, *shell_nprim, *shell_poff, *shell_ao;
    const double *pexp, *pcoef;
    double vmax;     // max_P N_P 2 pi / alpha_P
    double tol;      // <= 0: keep everything
};

constexpr int RIS_SCAN_BLOCK = 1024;

__device__ __forceinline__ void ris_decode_pair(long long t, int& i, int& j)
{
    long long r = (long long)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while (r * (r + 1) / 2 > t) --r;
    while ((r + 1) * (r + 2) / 2 <= t) ++r;
    i = (int)r;
    j = (int)(t - r * (r + 1) / 2);
}

// mu carries the larger l (ties: the larger shell index), so la >= lb in every class.
__device__ __forceinline__ void ris_order_pair(const RisMolDev& m, int i, int j, int& mu, int& nu)
{
    if (m.shell_l[i] >= m.shell_l[j]) { mu = i; nu = j; } else { mu = j; nu = i; }
}

__device__ __forceinline__ bool ris_prim_survives(const RisMolDev& m, double a, double b, double da, double db, double AB2)
{
    if (!(m.tol > 0.0)) return true;
    const double p = a + b;
    const double s = 3.14159265358979323846 / p;
    const double bound = fabs(da * db) * exp(-a * b / p * AB2) * s * sqrt(s) * m.vmax * (1.0 + 2.0 * fmax(a, b));
    return bound >= m.tol;
}

// Survey: packed[t] = cls | nkA << 8 | nkB << 20 with cls = 15 for a dropped pair; nkA / nkB = surviving
// primitive pairs hosted on A (a >= b) / on B (b > a).  Per-class max / total of surviving primitive pairs.
constexpr int RIS_NBIN = 16;
constexpr int RIS_DROPPED = 15;

// key[t] = cls << 40 | atom(mu) << 20 | atom(nu): the sort key (class, atom pair).
__global__ void __launch_bounds__(RIS_SCAN_BLOCK) ris_k_pair_survey(RisMolDev m, long long ntot, unsigned* packed,
                                                                    unsigned long long* key, int* kmax, unsigned long long* nprim)
{
    const long long t = (long long)blockIdx.x * RIS_SCAN_BLOCK + threadIdx.x;
    if (t >= ntot) return;
    int i, j, mu, nu;
    ris_decode_pair(t, i, j);
    ris_order_pair(m, i, j, mu, nu);
    const double* A = m.coords + 3 * m.shell_atom[mu];
    const double* B = m.coords + 3 * m.shell_atom[nu];
    const double dx = A[0] - B[0], dy = A[1] - B[1], dz = A[2] - B[2];
    const double AB2 = dx * dx + dy * dy + dz * dz;
    // (l,s) pairs are hosted on the l shell (mu) for every primitive pair: nothing is transferred by the HRR, the derivative
    // with respect to the s centre is a direct recurrence step there (gen_classes.py) -- one phase per pair
    const bool ss = m.shell_l[nu] == 0;
    int nA = 0, nB = 0;
    for (int ka = 0; ka < m.shell_nprim[mu]; ++ka)
        for (int kb = 0; kb < m.shell_nprim[nu]; ++kb) {
            const double a = m.pexp[m.shell_poff[mu] + ka], b = m.pexp[m.shell_poff[nu] + kb];
            if (!ris_prim_survives(m, a, b, m.pcoef[m.shell_poff[mu] + ka], m.pcoef[m.shell_poff[nu] + kb], AB2)) continue;
            if (a >= b || ss) ++nA; else ++nB;
        }
    unsigned k = RIS_DROPPED;
    if (nA + nB > 0) {
        k = (unsigned)ris_class_id(m.shell_l[mu], m.shell_l[nu]);
        atomicMax(&kmax[k], nA + nB);
        atomicAdd(&nprim[k], (unsigned long long)(nA + nB));
    }
    packed[t] = k | ((unsigned)min(nA, 4095) << 8) | ((unsigned)min(nB, 4095) << 20);
    key[t] = ((unsigned long long)k << 40) | ((unsigned long long)m.shell_atom[mu] << 20) | (unsigned long long)m.shell_atom[nu];
}

// Stable LSD radix sort of the pair list on 4-bit digits of the key (atom of nu, atom of mu, class; `shift` selects
// the digit).  After it the pairs of a class are contiguous and ordered by atom pair: the class kernel walks the shell
// pairs of one atom pair back to back and keeps their pair-side gradient in registers.
__device__ __forceinline__ int ris_digit(unsigned long long key, int shift) { return (int)((key >> shift) & 15ull); }

__global__ void __launch_bounds__(RIS_SCAN_BLOCK) ris_k_radix_hist(long long n, const long long* list_in, const unsigned long long* key,
                                                                   int shift, int* hist)
{
    __shared__ int sh[RIS_NBIN];
    if (threadIdx.x < RIS_NBIN) sh[threadIdx.x] = 0;
    __syncthreads();
    const long long i = (long long)blockIdx.x * RIS_SCAN_BLOCK + threadIdx.x;
    if (i < n) atomicAdd(&sh[ris_digit(key[list_in ? list_in[i] : i], shift)], 1);
    __syncthreads();
    if (threadIdx.x < RIS_NBIN) hist[blockIdx.x * RIS_NBIN + threadIdx.x] = sh[threadIdx.x];
}

// Exclusive scan over blocks for each bin -> base[blk][bin]; totals[bin]; start[bin] (bin-major order).
// One block of RIS_NBIN warps, warp c = bin c: every lane sums a contiguous run of blocks (independent loads), the lane sums
// are scanned with shuffles, a second pass writes the bases.  (One thread per bin walking all blocks took 0.27 ms per pass
// at config 4 -- 3562 blocks, 7 passes: two thirds of the kernel time of ris_setup.)
__global__ void __launch_bounds__(32 * RIS_NBIN) ris_k_radix_scan(int nblk, const int* hist, int* base, int* totals, int* start)
{
    __shared__ int tot[RIS_NBIN];
    const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int per = (nblk + 31) / 32;
    const int b0 = min(lane * per, nblk), b1 = min(b0 + per, nblk);
    int sum = 0;
#pragma unroll 4
    for (int b = b0; b < b1; ++b) sum += hist[b * RIS_NBIN + c];
    int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    int run = incl - sum;
    for (int b = b0; b < b1; ++b) { base[b * RIS_NBIN + c] = run; run += hist[b * RIS_NBIN + c]; }
    if (lane == 31) { totals[c] = incl; tot[c] = incl; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int r = 0;
        for (int k = 0; k < RIS_NBIN; ++k) { start[k] = r; r += tot[k]; }
    }
}

// Stable scatter: list_out[start[d] + base[blk][d] + rank-in-block] = element.
__global__ void __launch_bounds__(RIS_SCAN_BLOCK) ris_k_radix_scatter(long long n, const long long* list_in, const unsigned long long* key,
                                                                      int shift, const int* base, const int* start, long long* list_out)
{
    __shared__ int wtot[RIS_SCAN_BLOCK / 32];
    const long long i = (long long)blockIdx.x * RIS_SCAN_BLOCK + threadIdx.x;
    const long long el = (i < n) ? (list_in ? list_in[i] : i) : -1;
    const int k = (i < n) ? ris_digit(key[el], shift) : -1;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int c = 0; c < RIS_NBIN; ++c) {
        const unsigned bal = __ballot_sync(0xffffffffu, k == c);
        if (lane == 0) wtot[w] = __popc(bal);
        __syncthreads();
        if (k == c) {
            int rank = __popc(bal & ((1u << lane) - 1u));
            for (int ww = 0; ww < w; ++ww) rank += wtot[ww];
            list_out[start[c] + base[blockIdx.x * RIS_NBIN + c] + rank] = el;
        }
        __syncthreads();
    }
}

// prim_off[0 .. n] = exclusive scan of the surviving primitive-pair counts of the class's sorted pairs (one block).
__global__ void __launch_bounds__(1024) ris_k_scan_nk(int n, const long long* list, const unsigned* packed, long long* prim_off)
{
    __shared__ long long part[1024];
    const int t = threadIdx.x, per = (n + 1023) / 1024;
    const int i0 = min(t * per, n), i1 = min(i0 + per, n);
    long long sum = 0;
    for (int i = i0; i < i1; ++i) { const unsigned pk = packed[list[i]]; sum += ((pk >> 8) & 4095u) + ((pk >> 20) & 4095u); }
    part[t] = sum;
    __syncthreads();
    if (t == 0) {
        long long run = 0;
        for (int k = 0; k < 1024; ++k) { const long long v = part[k]; part[k] = run; run += v; }
        prim_off[n] = run;
    }
    __syncthreads();
    long long run = part[t];
    for (int i = i0; i < i1; ++i) {
        prim_off[i] = run;
        const unsigned pk = packed[list[i]];
        run += ((pk >> 8) & 4095u) + ((pk >> 20) & 4095u);
    }
}

// task_begin[t] = first pair whose first primitive-pair record is >= t * task_prims  (t = 0 .. ntasks)
__global__ void ris_k_task_bounds(int npairs, int ntasks, int task_prims, const long long* prim_off, int* task_begin)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t > ntasks) return;
    const long long target = (long long)t * task_prims;
    int lo = 0, hi = npairs;             // first ip in [0, npairs] with prim_off[ip] >= target
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (prim_off[mid] >= target) hi = mid; else lo = mid + 1;
    }
    task_begin[t] = (t == ntasks) ? npairs : lo;
}

// Pack one class: pair records, AO offsets, symmetry factor, surviving primitive pairs -- those hosted on
// A (a >= b) first, then those hosted on B -- as 64-byte records at prim_off[ip].
__global__ void ris_k_pair_pack(RisMolDev m, RisClassPack pk, const long long* list)
{
    const int ip = blockIdx.x * blockDim.x + threadIdx.x;
    if (ip >= pk.npairs) return;
    int i, j, mu, nu;
    ris_decode_pair(list[ip], i, j);
    ris_order_pair(m, i, j, mu, nu);
    const int atA = m.shell_atom[mu], atB = m.shell_atom[nu];
    const double* A = m.coords + 3 * atA;
    const double* B = m.coords + 3 * atB;
    const double dx = A[0] - B[0], dy = A[1] - B[1], dz = A[2] - B[2];
    const double AB2 = dx * dx + dy * dy + dz * dz;
    const size_t n = (size_t)pk.npairs;
    RisPairRec rec;
    rec.Ax = A[0]; rec.Ay = A[1]; rec.Az = A[2];
    rec.ABx = dx; rec.ABy = dy; rec.ABz = dz;
    rec.atA = atA; rec.atB = atB;
    pk.ao[ip] = m.shell_ao[mu]; pk.ao[n + ip] = m.shell_ao[nu];
    pk.symf[ip] = (mu == nu) ? 0.5f : 1.0f;
    double* q = pk.prim + (size_t)pk.prim_off[ip] * RIS_PRIM_FIELDS;
    const bool ss = pk.lb == 0;
    int k = 0, kA = 0;
    for (int host = 0; host < 2; ++host) {
        for (int ka = 0; ka < m.shell_nprim[mu]; ++ka)
            for (int kb = 0; kb < m.shell_nprim[nu]; ++kb) {
                const double a = m.pexp[m.shell_poff[mu] + ka], b = m.pexp[m.shell_poff[nu] + kb];
                if ((a >= b || ss) != (host == 0)) continue;
                const double da = m.pcoef[m.shell_poff[mu] + ka], db = m.pcoef[m.shell_poff[nu] + kb];
                if (!ris_prim_survives(m, a, b, da, db, AB2)) continue;
                const double p = a + b, ip_ = 1.0 / p;
                q[0] = p;
                // P - Z (Z = host centre) from the centre difference: host A: -(b/p)(A-B); host B: (a/p)(A-B)
                const double fz = (host == 0) ? -b * ip_ : a * ip_;
                q[1] = fz * dx;
                q[2] = fz * dy;
                q[3] = fz * dz;
                q[4] = 0.5 * ip_;
                q[5] = 2.0 * a;
                q[6] = 2.0 * b;
                // d_a d_b K_ab 2 pi^{5/2} / p
                q[7] = da * db * exp(-a * b * ip_ * AB2) * (2.0 * 17.493418327624862846) * ip_;
                q += RIS_PRIM_FIELDS;
                ++k;
            }
        if (host == 0) kA = k;
    }
    rec.nkA = kA; rec.nkB = k - kA;
    pk.pairs[ip] = rec;
}
