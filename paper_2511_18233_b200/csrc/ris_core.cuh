// ris_core.cuh -- device-side arithmetic shared by the class kernels:
//   S1  Boys function F_m(T), m = 0..E
//   S2  one primitive triplet: prefactor, Boys, OS recurrence
// The integrals are (pq|A) of Eq. 21 and their nuclear derivatives, Eq. 27 terms 1-2
// (PAPER.md:119, 150); the paper does not describe their evaluation.
#pragma once
#include <math.h>
#include <stddef.h>

#ifndef RIS_DEV
#define RIS_DEV __device__ __forceinline__
#endif

template <int LA, int LB> struct RisClass;
template <int LA, int LB> struct RisClass0;     // undifferentiated integrals (fitting step)
#include "generated/ris_classes.cuh"

// ---------------------------------------------------------------------------------------------
// Boys function.
//   T < RIS_BOYS_TMAX: nearest grid point T0 = i/32, x = T - T0 in [-1/64, 1/64];
//       F_M(T)  = sum_{k=0..6} F_{M+k}(T0) (-x)^k / k!      (Taylor; d/dT F_m = -F_{m+1})
//       e^{-T}  = e^{-T0} sum_{k=0..6} (-x)^k / k!
//       F_m     = (2T F_{m+1} + e^{-T}) / (2m+1)             (downward, stable)
//     truncation < (1/64)^7/7! = 4.4e-17 relative.  One table row per grid point and per top
//     order M: {e^{-T0}, c_0..c_6}, c_k = (-1)^k F_{M+k}(T0)/k!  (64 bytes, one 2-sector gather).
//   T >= RIS_BOYS_TMAX (=40): erfc(sqrt T) < 4e-19, so F_0 = sqrt(pi/T)/2, and upward
//       F_{m+1} = ((2m+1) F_m - e^{-T}) / (2T)
//     where e^{-T} is at most a 6e-11 relative correction (m = 7, T = 40): single precision is enough.
constexpr double RIS_BOYS_TMAX = 40.0;
constexpr int RIS_BOYS_PER_UNIT = 32;
constexpr int RIS_BOYS_NGRID = 40 * 32 + 1;
constexpr int RIS_BOYS_ROW = 8;

// 1/sqrt(x) for positive, normal x (p + alpha, T >= 40), branch-free: the hardware seed (MUFU.RSQ64H, relative error
// < 2^-22) and ONE third-order step  y (1 + e/2 + 3 e^2/8),  e = 1 - x y^2  (error ~ e^3 = 2^-66; the result is within an
// ulp or two of the correctly rounded value).  CUDA's rsqrt() adds special-case branches this path never needs.
RIS_DEV double ris_rsqrt(double x)
{
#ifdef __CUDA_ARCH__
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-(x * y), y, 1.0);
    return fma(y * e, fma(0.375, e, 0.5), y);
#else
    return 1.0 / sqrt(x);
#endif
}

// e^{-T} for T >= 40, single precision (see the error budget above): one FMUL + MUFU.EX2
RIS_DEV double ris_exp_neg_f32(double T)
{
#ifdef __CUDA_ARCH__
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(-1.44269504088896340736f * (float)T));
    return (double)r;
#else
    return (double)expf(-(float)T);
#endif
}

// F[m] = scale * F_m(T), m = 0..M.  The scale (kappa of the primitive triplet) rides along: the recursions are linear
// in (F, e^{-T}), so two multiplications replace M + 1.
template <int M>
RIS_DEV void ris_boys(double T, const double* __restrict__ tab, double (&F)[M + 1], double scale = 1.0)
{
    if (T < RIS_BOYS_TMAX) {
        const int i = (int)(T * RIS_BOYS_PER_UNIT + 0.5);
        const double x = T - (double)i * (1.0 / RIS_BOYS_PER_UNIT);
        const double* __restrict__ r = tab + (size_t)i * RIS_BOYS_ROW;
#ifdef __CUDA_ARCH__
        const double2 r0 = __ldg(reinterpret_cast<const double2*>(r));
        const double2 r1 = __ldg(reinterpret_cast<const double2*>(r) + 1);
        const double2 r2 = __ldg(reinterpret_cast<const double2*>(r) + 2);
        const double2 r3 = __ldg(reinterpret_cast<const double2*>(r) + 3);
        const double e0 = r0.x, c0 = r0.y, c1 = r1.x, c2 = r1.y, c3 = r2.x, c4 = r2.y, c5 = r3.x, c6 = r3.y;
#else
        const double e0 = r[0], c0 = r[1], c1 = r[2], c2 = r[3], c3 = r[4], c4 = r[5], c5 = r[6], c6 = r[7];
#endif
        double f = fma(c6, x, c5);
        f = fma(f, x, c4);
        f = fma(f, x, c3);
        f = fma(f, x, c2);
        f = fma(f, x, c1);
        f = fma(f, x, c0);
        double ex = fma(x, 1.0 / 720.0, -1.0 / 120.0);
        ex = fma(ex, x, 1.0 / 24.0);
        ex = fma(ex, x, -1.0 / 6.0);
        ex = fma(ex, x, 0.5);
        ex = fma(ex, x, -1.0);
        ex = fma(ex, x, 1.0);
        ex *= e0 * scale;
        f *= scale;
        F[M] = f;
        const double t2 = T + T;
#pragma unroll
        for (int m = M - 1; m >= 0; --m) {
            f = fma(t2, f, ex) * (1.0 / (2 * m + 1));
            F[m] = f;
        }
    } else {
        const double rt = ris_rsqrt(T);
        const double i2t = 0.5 * rt * rt;
        const double ex = ris_exp_neg_f32(T) * scale;
        double f = (0.88622692545275801365 * scale) * rt;     // sqrt(pi)/2 / sqrt(T)
        F[0] = f;
#pragma unroll
        for (int m = 0; m < M; ++m) {
            f = fma((double)(2 * m + 1), f, -ex) * i2t;
            F[m + 1] = f;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// One primitive triplet (primitive of mu, primitive of nu, aux P), hosted on centre Z (see gen_classes.py:
// Z = A for primitive pairs with a >= b, Z = B otherwise; LH/LO are the host's / the other shell's l):
//   rho = p alpha/(p+alpha), T = rho |P-C|^2, [0]^(m) = kappa F_m(T) with
//   kappa = coef * auxfac / sqrt(p+alpha),  coef = d_a d_b K_ab 2 pi^{5/2}/p,  auxfac = N_P/alpha,
// then the class recurrence + exponent-scaled accumulation (generated code); h2 / o2 = 2 x exponent of the
// host / other primitive.
// Accuracy: the packed record carries PZ = P - Z = -(o/p)(Z - O) computed from the centre difference, never
// as a difference of absolute coordinates: for a tight pair on one atom the whole derivative is the small
// WP term, and a rounding residue of size eps*|coords| in P - Z would swamp it.  P - C = (Z - C) + PZ.
// Split in two so the class kernel can software-pipeline the primitive loop: ris_prim_head (prefactor + Boys: one
// long dependent chain through rsqrt, the table gather and two Horner schemes) of primitive k+1 is issued next to
// the wide, independent recurrence of primitive k.
template <int E>
struct RisPrimHead {
    double F[E + 1];          // kappa F_m(T)
    double W0, W1, W2;        // W - P = -(rho/p)(P - C)
    double q;                 // rho/p
};

template <int E>
RIS_DEV void ris_prim_head(double p, double PZx, double PZy, double PZz, double coef, double ZCx, double ZCy, double ZCz,
                           double alpha, double auxfac, const double* __restrict__ boys_tab, RisPrimHead<E>& h)
{
    const double s = ris_rsqrt(p + alpha);
    const double q = alpha * s * s;          // rho/p
    const double X0 = ZCx + PZx, X1 = ZCy + PZy, X2 = ZCz + PZz;
    const double T = (p * q) * fma(X0, X0, fma(X1, X1, X2 * X2));
    ris_boys<E>(T, boys_tab, h.F, (coef * auxfac) * s);
    h.W0 = -q * X0; h.W1 = -q * X1; h.W2 = -q * X2;
    h.q = q;
}

// The branch-free front of the head (everything before the Boys function), used by the software-pipelined primitive
// loop of the class kernel: it is issued for primitive k+1 next to the recurrence of primitive k.
struct RisPrimFront {
    double T, kappa, q, X0, X1, X2;       // rho |P-C|^2, coef auxfac / sqrt(p+alpha), rho/p, P - C
};

RIS_DEV void ris_prim_front(double p, double PZx, double PZy, double PZz, double coef, double ZCx, double ZCy, double ZCz,
                            double alpha, double auxfac, RisPrimFront& f)
{
    const double s = ris_rsqrt(p + alpha);
    f.q = alpha * s * s;
    f.X0 = ZCx + PZx; f.X1 = ZCy + PZy; f.X2 = ZCz + PZz;
    f.T = (p * f.q) * fma(f.X0, f.X0, fma(f.X1, f.X1, f.X2 * f.X2));
    f.kappa = (coef * auxfac) * s;
}

// plain-memory tile provider of the generated contraction code (the class kernel passes its shared-memory ring instead)
struct RisTilePlain {
    const double* tile; size_t estride, sstride;
    RIS_DEV size_t es() const { return estride; }
    RIS_DEV const double* get(int s) const { return tile + (size_t)s * sstride; }
};

// ZO = Z - O (host centre minus other centre).  Classes with an s function on the other centre (LO = 0) take the derivative
// with respect to it by a direct recurrence step there (gen_classes.py): P - O = (h/p)(Z - O), from the exponents.
template <int LH, int LO, class ACC>
RIS_DEV void ris_prim_triplet(double p, double PZx, double PZy, double PZz, double oo2p, double h2, double o2,
                              double coef, double ZCx, double ZCy, double ZCz, double alpha, double auxfac,
                              const double* __restrict__ boys_tab, ACC& acc, double ZOx, double ZOy, double ZOz)
{
    constexpr int E = RisClass<LH, LO>::E;
    RisPrimHead<E> h;
    ris_prim_head<E>(p, PZx, PZy, PZz, coef, ZCx, ZCy, ZCz, alpha, auxfac, boys_tab, h);
    if constexpr (LO == 0) {
        const double hp = h2 * oo2p;
        ris_vrr<LH, LO>(h.F, PZx, PZy, PZz, h.W0, h.W1, h.W2, oo2p, h.q, h2, o2, acc, hp * ZOx, hp * ZOy, hp * ZOz);
    } else {
        ris_vrr<LH, LO>(h.F, PZx, PZy, PZz, h.W0, h.W1, h.W2, oo2p, h.q, h2, o2, acc);
    }
}

// p-type auxiliary function, component DIR (NEXT-2): the s-aux ladder one Boys order higher, then one
// recurrence step on the aux centre (gen_classes.py "p-type auxiliary functions"): WC = (W - C)_DIR = (1 - rho/p)(P - C)_DIR,
// 1/(2(p + alpha)) = (rho/p)/(2 alpha).  boys_tab: the table of order E + 1.
template <int LH, int LO, int DIR, class ACC>
RIS_DEV void ris_prim_triplet_p(double p, double PZx, double PZy, double PZz, double oo2p, double h2, double o2,
                                double coef, double ZCx, double ZCy, double ZCz, double alpha, double auxfac,
                                const double* __restrict__ boys_tab, ACC& acc, double ZOx, double ZOy, double ZOz)
{
    constexpr int E = RisClass<LH, LO>::E;
    RisPrimHead<E + 1> h;
    ris_prim_head<E + 1>(p, PZx, PZy, PZz, coef, ZCx, ZCy, ZCz, alpha, auxfac, boys_tab, h);
    const double X = DIR == 0 ? ZCx + PZx : (DIR == 1 ? ZCy + PZy : ZCz + PZz);
    const double WC = (1.0 - h.q) * X, oo2pa = 0.5 * h.q / alpha;
    if constexpr (LO == 0) {
        const double hp = h2 * oo2p;
        ris_vrrp<LH, LO, DIR>(h.F, PZx, PZy, PZz, h.W0, h.W1, h.W2, oo2p, h.q, h2, o2, acc, WC, oo2pa, hp * ZOx, hp * ZOy, hp * ZOz);
    } else {
        ris_vrrp<LH, LO, DIR>(h.F, PZx, PZy, PZz, h.W0, h.W1, h.W2, oo2p, h.q, h2, o2, acc, WC, oo2pa);
    }
}

template <int LH, int LO, int DIR>
RIS_DEV void ris_prim_triplet0_p(double p, double PZx, double PZy, double PZz, double oo2p, double coef, double ZCx,
                                 double ZCy, double ZCz, double alpha, double auxfac, const double* __restrict__ boys_tab,
                                 double (&acc)[RisClass0<LH, LO>::NACC])
{
    constexpr int E = RisClass0<LH, LO>::E;
    RisPrimHead<E + 1> h;
    ris_prim_head<E + 1>(p, PZx, PZy, PZz, coef, ZCx, ZCy, ZCz, alpha, auxfac, boys_tab, h);
    const double X = DIR == 0 ? ZCx + PZx : (DIR == 1 ? ZCy + PZy : ZCz + PZz);
    ris_vrrp0<LH, LO, DIR>(h.F, PZx, PZy, PZz, h.W0, h.W1, h.W2, oo2p, h.q, 0.0, 0.0, acc, (1.0 - h.q) * X, 0.5 * h.q / alpha);
}

// Undifferentiated primitive triplet (v_P = sum D_{mu nu} (mu nu|P), Eq. 21):
// the same head, the VRR up to e = lh + lo, unscaled accumulation of [e0|s].
template <int LH, int LO>
RIS_DEV void ris_prim_triplet0(double p, double PZx, double PZy, double PZz, double oo2p, double coef, double ZCx,
                               double ZCy, double ZCz, double alpha, double auxfac, const double* __restrict__ boys_tab,
                               double (&acc)[RisClass0<LH, LO>::NACC])
{
    constexpr int E = RisClass0<LH, LO>::E;
    RisPrimHead<E> h;
    ris_prim_head<E>(p, PZx, PZy, PZz, coef, ZCx, ZCy, ZCz, alpha, auxfac, boys_tab, h);
    ris_vrr0<LH, LO>(h.F, PZx, PZy, PZz, h.W0, h.W1, h.W2, oo2p, h.q, 0.0, 0.0, acc);
}
