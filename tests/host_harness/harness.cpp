// Host-side test harness (tests only, never part of the product path): compiles the generated class
// recurrences and the Boys interpolation of paper_2511_18233_b200/csrc as plain C++ so that the CPU
// test-suite can check their arithmetic against the oracle without a GPU.
#define RIS_DEV inline
#include "ris_core.cuh"
#include "ris_boys_table.h"
#include <cstring>
#include <map>
#include <vector>

static std::map<int, std::vector<double>> g_tabs;
static const double* tab(int M)
{
    auto it = g_tabs.find(M);
    if (it == g_tabs.end()) {
        std::vector<double> t;
        ris_build_boys_table(M, RIS_BOYS_NGRID, RIS_BOYS_PER_UNIT, t);
        it = g_tabs.emplace(M, std::move(t)).first;
    }
    return it->second.data();
}

template <int M> static void boys_t(double T, double* F)
{
    double f[M + 1];
    ris_boys<M>(T, tab(M), f);
    for (int m = 0; m <= M; ++m) F[m] = f[m];
}

extern "C" int harness_boys(int M, double T, double* F)
{
    switch (M) {
    case 0: boys_t<0>(T, F); break;
    case 1: boys_t<1>(T, F); break; case 2: boys_t<2>(T, F); break; case 3: boys_t<3>(T, F); break;
    case 4: boys_t<4>(T, F); break; case 5: boys_t<5>(T, F); break; case 6: boys_t<6>(T, F); break;
    case 7: boys_t<7>(T, F); break; case 8: boys_t<8>(T, F); break; default: return -1;
    }
    return 0;
}

// One contracted triplet: nk primitive pairs (prim[k][8] = p,(P-Z)x,(P-Z)y,(P-Z)z,oo2p,a2,b2,coef; Z = host centre), aux (C, alpha,
// auxfac); tile[nb][nca*ncb]; out[nb][6] = (dA, dB) contracted with the tile.  Primitive pairs with a >= b
// are hosted on A, the others on B, exactly as the class kernel does.
// AUX: 0 = s-type auxiliary function, 1..3 = p_x, p_y, p_z (NEXT-2)
template <int LH, int LO, bool TR, int AUX>
static void phase_t(int nk, const double* prim, bool hostA, const double* Z, const double* ZO, const double* C,
                    double alpha, double auxfac, const double* tile, int nb, double* out)
{
    using K = RisClass<LH, LO>;
    // (l,s) pairs: every primitive pair is hosted on the l shell (ris_setup.cuh), whatever the exponents
    constexpr bool lb0 = TR ? (LH == 0) : (LO == 0);
    double acc[K::NACC];
    for (int i = 0; i < K::NACC; ++i) acc[i] = 0.0;
    int used = 0;
    for (int k = 0; k < nk; ++k) {
        const double* q = prim + 8 * k;
        if ((q[5] >= q[6] || lb0) != hostA) continue;
        ++used;
        if constexpr (AUX == 0)
            ris_prim_triplet<LH, LO>(q[0], q[1], q[2], q[3], q[4], hostA ? q[5] : q[6], hostA ? q[6] : q[5], q[7],
                                     Z[0] - C[0], Z[1] - C[1], Z[2] - C[2], alpha, auxfac, tab(K::E), acc, Z[0] - ZO[0], Z[1] - ZO[1],
                                     Z[2] - ZO[2]);
        else
            ris_prim_triplet_p<LH, LO, AUX - 1>(q[0], q[1], q[2], q[3], q[4], hostA ? q[5] : q[6], hostA ? q[6] : q[5], q[7],
                                                Z[0] - C[0], Z[1] - C[1], Z[2] - C[2], alpha, auxfac, tab(K::E + 1), acc,
                                                Z[0] - ZO[0], Z[1] - ZO[1], Z[2] - ZO[2]);
    }
    if (!used) return;
    // slots as in the class kernel: slot[(s*6 + c)*SL], c = 0..2 centre A, 3..5 centre B (stride SL = 1 here), unit scales
    std::vector<double> sc((size_t)nb, 1.0);
    RisTilePlain ring{tile, (size_t)1, (size_t)(K::NCA * K::NCB)};
    ris_hrrc<LH, LO, TR, 1, 1>(acc, Z[0] - ZO[0], Z[1] - ZO[1], Z[2] - ZO[2], ring, nb, sc.data(), out);
}

template <int LA, int LB, int AUX>
static void triplet_t(int nk, const double* prim, const double* A, const double* AB, const double* C, double alpha,
                      double auxfac, const double* tile, int nb, double* out)
{
    const double B[3] = {A[0] - AB[0], A[1] - AB[1], A[2] - AB[2]};
    for (int i = 0; i < 6 * nb; ++i) out[i] = 0.0;
    phase_t<LA, LB, false, AUX>(nk, prim, true, A, B, C, alpha, auxfac, tile, nb, out);
    phase_t<LB, LA, true, AUX>(nk, prim, false, B, A, C, alpha, auxfac, tile, nb, out);
}

extern "C" int harness_triplet_aux(int la, int lb, int aux, int nk, const double* prim, const double* A, const double* AB,
                                   const double* C, double alpha, double auxfac, const double* tile, int nb, double* out)
{
#define CASE(a, b)                                                                                                     \
    if (la == a && lb == b) {                                                                                          \
        if (aux == 0) triplet_t<a, b, 0>(nk, prim, A, AB, C, alpha, auxfac, tile, nb, out);                            \
        else if (aux == 1) triplet_t<a, b, 1>(nk, prim, A, AB, C, alpha, auxfac, tile, nb, out);                       \
        else if (aux == 2) triplet_t<a, b, 2>(nk, prim, A, AB, C, alpha, auxfac, tile, nb, out);                       \
        else if (aux == 3) triplet_t<a, b, 3>(nk, prim, A, AB, C, alpha, auxfac, tile, nb, out);                       \
        else return -1;                                                                                                \
        return 0;                                                                                                      \
    }
    CASE(0, 0) CASE(1, 0) CASE(1, 1) CASE(2, 0) CASE(2, 1) CASE(2, 2) CASE(3, 0) CASE(3, 1) CASE(3, 2) CASE(3, 3)
#undef CASE
    return -1;
}

extern "C" int harness_triplet(int la, int lb, int nk, const double* prim, const double* A, const double* AB,
                               const double* C, double alpha, double auxfac, const double* tile, int nb, double* out)
{
    return harness_triplet_aux(la, lb, 0, nk, prim, A, AB, C, alpha, auxfac, tile, nb, out);
}

// The undifferentiated contracted triplet (fitting step): out[nb] = sum_{ab} tile[s][a][b] (ab|P), phases as above.
template <int LH, int LO, bool TR, int AUX>
static void phase0_t(int nk, const double* prim, bool hostA, const double* Z, const double* ZO, const double* C,
                     double alpha, double auxfac, const double* tile, int nb, int nel, double* out)
{
    using K = RisClass0<LH, LO>;
    constexpr bool lb0 = TR ? (LH == 0) : (LO == 0);
    double acc[K::NACC];
    for (int i = 0; i < K::NACC; ++i) acc[i] = 0.0;
    int used = 0;
    for (int k = 0; k < nk; ++k) {
        const double* q = prim + 8 * k;
        if ((q[5] >= q[6] || lb0) != hostA) continue;
        ++used;
        if constexpr (AUX == 0)
            ris_prim_triplet0<LH, LO>(q[0], q[1], q[2], q[3], q[4], q[7], Z[0] - C[0], Z[1] - C[1], Z[2] - C[2], alpha, auxfac,
                                      tab(K::E), acc);
        else
            ris_prim_triplet0_p<LH, LO, AUX - 1>(q[0], q[1], q[2], q[3], q[4], q[7], Z[0] - C[0], Z[1] - C[1], Z[2] - C[2], alpha,
                                                 auxfac, tab(K::E + 1), acc);
    }
    if (!used) return;
    ris_hrr0c<LH, LO, TR, 1>(acc, Z[0] - ZO[0], Z[1] - ZO[1], Z[2] - ZO[2], tile, (size_t)1, (size_t)nel, nb, out);
}

template <int LA, int LB, int AUX>
static void triplet0_t(int nk, const double* prim, const double* A, const double* AB, const double* C, double alpha,
                       double auxfac, const double* tile, int nb, double* out)
{
    const double B[3] = {A[0] - AB[0], A[1] - AB[1], A[2] - AB[2]};
    constexpr int nel = RisClass<LA, LB>::NCA * RisClass<LA, LB>::NCB;
    for (int i = 0; i < nb; ++i) out[i] = 0.0;
    phase0_t<LA, LB, false, AUX>(nk, prim, true, A, B, C, alpha, auxfac, tile, nb, nel, out);
    phase0_t<LB, LA, true, AUX>(nk, prim, false, B, A, C, alpha, auxfac, tile, nb, nel, out);
}

extern "C" int harness_triplet0_aux(int la, int lb, int aux, int nk, const double* prim, const double* A, const double* AB,
                                    const double* C, double alpha, double auxfac, const double* tile, int nb, double* out)
{
#define CASE(a, b)                                                                                                     \
    if (la == a && lb == b) {                                                                                          \
        if (aux == 0) triplet0_t<a, b, 0>(nk, prim, A, AB, C, alpha, auxfac, tile, nb, out);                           \
        else if (aux == 1) triplet0_t<a, b, 1>(nk, prim, A, AB, C, alpha, auxfac, tile, nb, out);                      \
        else if (aux == 2) triplet0_t<a, b, 2>(nk, prim, A, AB, C, alpha, auxfac, tile, nb, out);                      \
        else if (aux == 3) triplet0_t<a, b, 3>(nk, prim, A, AB, C, alpha, auxfac, tile, nb, out);                      \
        else return -1;                                                                                                \
        return 0;                                                                                                      \
    }
    CASE(0, 0) CASE(1, 0) CASE(1, 1) CASE(2, 0) CASE(2, 1) CASE(2, 2) CASE(3, 0) CASE(3, 1) CASE(3, 2) CASE(3, 3)
#undef CASE
    return -1;
}

extern "C" int harness_triplet0(int la, int lb, int nk, const double* prim, const double* A, const double* AB,
                                const double* C, double alpha, double auxfac, const double* tile, int nb, double* out)
{
    return harness_triplet0_aux(la, lb, 0, nk, prim, A, AB, C, alpha, auxfac, tile, nb, out);
}
