// ris_grad_kernel.cuh -- the fused class kernel: S1 Boys + S2 derivative-integral recurrence +
// S3 contraction with the D / Gamma^P tile + S4 reduction, one instantiation per
// (l_mu,l_nu) class and contraction type.  Eq. 27 terms 1-2 for the integrals of Eq. 21
// (PAPER.md:119).
//
// Mapping ("aux lanes"): the 32 lanes of a warp hold 32 different auxiliary functions P (blockIdx.y selects the
// chunk of 32) and walk TOGETHER through the shell pairs of a warp task (a window of packed primitive pairs,
// ris_internal.h).  Everything that belongs to the shell pair -- pair record, primitive-pair records, loop trip counts,
// the host-centre phases, the D tile of the J term -- is therefore warp-uniform: it is staged once per task into the
// warp's shared memory with coalesced 16-byte copies and read back as broadcasts, there is no divergence except the
// Boys-function branch, and what varies per lane (aux centre / exponent, W - P, Boys values, the Gamma^P tile of the
// K term, stored P-minor so a warp reads 256 contiguous bytes per element) is exactly the per-lane arithmetic.
//
// Tile staging (north_star: "shared-memory staging of D/Gamma tiles"): the pair's tile -- K: NEL rows of 32 aux values per
// state, J: NEL values per state -- is copied global -> shared with cp.async (LDGSTS) at the START of the pair, state by
// state into a ring of NS slots, and is waited for only when the contraction of that state begins: the DRAM / L2 latency
// of the Gamma^P read runs under the primitive loop (profiles/r01_v9_ncu.md: the K kernels lost 10-15 % to
// long_scoreboard stalls on these loads, (2,2) 78 %).
//
// Primitive loop: software-pipelined by hand -- the record load and the branch-free front of the prefactor chain
// (rsqrt(p + alpha), T) of primitive k+1 are issued next to the wide recurrence of primitive k.
//
// The per-state gradient accumulators are per-lane shared-memory slots (conflict-free: lane-contiguous), which keeps the
// register file for the recurrence:
//   aux side   g[A_P] = -(dA + dB) summed over the pairs (translational invariance): the lane owns P, so this is one
//              slot per (state, x) over ALL tasks of the warp; the warps of a block (same P chunk) are summed
//              in fixed order at the end, one atomic per (block, P, state, x).
//   pair side  g[A_mu], g[A_nu]: slots across the consecutive shell pairs of one atom pair (the pairs of a class
//              are sorted by atom pair), then a fixed-order sum over the lanes and one atomic per (atom pair, state,
//              centre, x).
// Every in-block sum has a fixed order; the global atomics are FP64 adds, or -- deterministic mode -- 64-bit integer
// adds of a fixed-point split (ris_grad_add), which makes the result bitwise reproducible.
#pragma once
#include "ris_core.cuh"
#include "ris_internal.h"
#include <type_traits>

// ------------------------------------------------------------------------------------------------ tuning
// resident blocks per SM the register allocation aims at (light classes: latency-bound prefactor / Boys chains
// want warps; heavy classes: the contracted targets want registers)
#ifndef RIS_MB1
#define RIS_MB1 4
#define RIS_MB2 3
#define RIS_MB3 2
#define RIS_MB4 2
#endif
// SPLIT: the heavy classes (l_mu + l_nu >= 4) run their two host-centre phases as two launches (PH = 1: primitive pairs
// hosted on A, PH = 2: hosted on B; PH = 0: both in one kernel).  With both phases inlined the (2,2) kernel is 94 KB of
// SASS and stalls on instruction fetch; one phase is 47 KB.
#ifndef RIS_PIPE_L
#define RIS_PIPE_L -1           // software-pipelined primitive loop for l_mu + l_nu <= this.  Measured on config 4 (r02):
#endif                          // slower for every class ((1,0) J 0.78 -> 0.92 ms): the extra live front spills at the
                                // register caps below and the last front of a phase is wasted -- off
#ifndef RIS_NSK2_BYTES
#define RIS_NSK2_BYTES 16384    // two ring slots at least when they take no more than this per warp.  (2,2) runs ONE 9 KB slot:
#endif                          // with two, the ring crowds the local-memory spills of that class out of L1 (K 0.57 -> 0.51 ms)
#ifndef RIS_STAGE_BYTES
#define RIS_STAGE_BYTES 13824   // shared-memory budget per warp for the K tile ring: three states of the (2,1) class (18 rows of
                                // 256 bytes each), so that the usual batch of <= 3 states has a slot per state (fast path of get)
#endif
template <int LA, int LB> struct RisGradTune {
    static constexpr int MINB = (LA + LB <= 1) ? RIS_MB1 : (LA + LB == 2 ? RIS_MB2 : (LA + LB == 3 ? RIS_MB3 : RIS_MB4));
    static constexpr bool SPLIT = ris_grad_split(LA, LB);
    static constexpr bool PIPE = (LA + LB <= RIS_PIPE_L);
    static constexpr int NEL = RisClass<LA, LB>::NCA * RisClass<LA, LB>::NCB;
    // slots of the tile ring: K -- as many states as fit the budget, at least 2 (1 for (2,2) and the f classes, whose slot
    // is 9-26 KB per warp), at most RIS_NB_MAX; J -- all states (a few doubles each)
    static constexpr int NSK_LO = (NEL * 256 * 2 <= RIS_NSK2_BYTES) ? 2 : 1;
    static constexpr int NSK = (RIS_STAGE_BYTES / (NEL * 256) < NSK_LO) ? NSK_LO
                             : (RIS_STAGE_BYTES / (NEL * 256) > RIS_NB_MAX ? RIS_NB_MAX : RIS_STAGE_BYTES / (NEL * 256));
    static constexpr bool STAGE_K = ris_grad_stage_k(LA, LB);      // else the K tile is read straight from global memory
    static constexpr int NW = RIS_GRAD_WARPS;                      // warps per block
};
// doubles of a tile ring of ns slots: K -- slots of NEL rows of 32 aux values; J -- slots of NEL values
template <int LA, int LB, bool KT> __host__ __device__ constexpr int ris_grad_tile_doubles(int ns)
{
    return KT ? (RisGradTune<LA, LB>::STAGE_K ? ns * RisGradTune<LA, LB>::NEL * 32 : 0) : ((ns * RisGradTune<LA, LB>::NEL + 1) & ~1);
}

// ------------------------------------------------------------------------------------------------ tile ring
__device__ __forceinline__ void ris_cp_async8(double* dst, const double* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void ris_cp_async16(double* dst, const double* src, int src_bytes)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void ris_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void ris_cp_wait(int pending)       // pending = groups that may still be in flight (0..4)
{
    switch (pending) {
    case 0: asm volatile("cp.async.wait_group 0;" ::: "memory"); break;
    case 1: asm volatile("cp.async.wait_group 1;" ::: "memory"); break;
    case 2: asm volatile("cp.async.wait_group 2;" ::: "memory"); break;
    case 3: asm volatile("cp.async.wait_group 3;" ::: "memory"); break;
    default: asm volatile("cp.async.wait_group 4;" ::: "memory"); break;
    }
}

// The staged tile of ONE shell pair.  State s lives in slot s % NS; get(s) returns the lane's view of it
// (element el at ptr[el * ES]) after its copy has landed, and refills the slot the previous state left.
//   K (KT): slot = [NEL][32] doubles, one 256-byte row per element (the 32 aux of this warp's chunk): two rows per
//           warp-wide 16-byte cp.async; rows of the last chunk are zero-filled beyond p1.
//   J:      slot = [NEL] doubles (the same for every lane): one 8-byte cp.async per element.
template <int NEL, int NS, bool KT>
struct RisTileRing {
    static constexpr int SLOT = KT ? NEL * 32 : NEL;
    __device__ __forceinline__ constexpr size_t es() const { return KT ? 32 : 1; }
    double* buf;               // this warp's ring
    const double* g;           // K: tile + first element of the pair * estride + chunk offset; J: tile + first element
    size_t estride, sstride;
    int nb, ns, lane, nv;      // ns = min(nb, NS) slots in use; nv: valid aux functions of this warp's chunk (K)
    int issued;                // states whose copy has been issued (and committed) since begin()
    int rd;                    // slot of the state get() returned last

    __device__ __forceinline__ void issue_to(int s, int slot)
    {
        double* dst = buf + slot * SLOT;
        const double* src = g + (size_t)s * sstride;
        if (KT) {
            const int c2 = (lane & 15) * 2;
            const int bytes = min(max(nv - c2, 0), 2) * 8;
#pragma unroll
            for (int r = 0; r < NEL; r += 2) {
                const int row = r + (lane >> 4);
                if ((NEL & 1) == 0 || row < NEL) ris_cp_async16(dst + row * 32 + c2, src + (size_t)row * estride + c2, bytes);
            }
        } else {
#pragma unroll
            for (int e = 0; e < NEL; e += 32)
                if (e + lane < NEL) ris_cp_async8(dst + e + lane, src + e + lane);
        }
        ris_cp_commit();
    }
    // start of a pair (or of its second host phase when the ring does not hold all states): every lane has finished
    // reading the previous contents (the caller's __syncwarp)
    __device__ __forceinline__ void begin()
    {
        issued = 0;
        for (int s = 0; s < ns; ++s) issue_to(s, s);
        issued = ns;
    }
    __device__ __forceinline__ const double* get(int s)
    {
        if (nb <= ns) {
            // every state has a slot of its own (the usual case): the copies were issued at the start of the pair, a whole
            // primitive loop ago -- ONE wait for all of them at the first state, no refill, slot = state.  (The general path
            // below costs ~100 integer / branch instructions per state: slot arithmetic with a modulo, a jump table for the
            // immediate of cp.async.wait_group, the refill test; profiles/r02_v1_ncu.md: (0,0) ran 2.5 instructions per FP64 one.)
            if (s == 0) {
                asm volatile("cp.async.wait_all;" ::: "memory");
                __syncwarp();
            }
            return buf + s * SLOT + (KT ? lane : 0);
        }
        // states are asked for in order: rd = slot of state s, kept incrementally (s % ns without the division)
        if (s == 0) rd = 0;
        else {
            if (issued < nb) {           // issued == s - 1 + ns: the slot state s-1 leaves (rd) is the next one's, and it is
                __syncwarp();            // free once every lane is done with state s-1
                issue_to(issued, rd);
                ++issued;
            }
            rd = rd + 1 == ns ? 0 : rd + 1;
        }
        ris_cp_wait(issued - 1 - s);
        __syncwarp();
        return buf + rd * SLOT + (KT ? lane : 0);
    }
    __device__ __forceinline__ bool holds_all() const { return nb <= ns; }
};

// Unstaged K tile (the 60- and 100-element classes): the same interface on global memory, element el of state s of this
// lane's aux function at g[s * sstride + el * estride].
struct RisTileDirectK {
    const double* g;           // tile + first element of the pair * estride + chunk offset (set per pair)
    size_t estride, sstride;
    int nb, ns, lane, nv, issued;
    __device__ __forceinline__ size_t es() const { return estride; }
    __device__ __forceinline__ void begin() {}
    __device__ __forceinline__ const double* get(int s) const { return g + (size_t)s * sstride + (lane < nv ? lane : 0); }
    __device__ __forceinline__ bool holds_all() const { return true; }
};

// ------------------------------------------------------------------------------------------------ one host-centre phase
// The primitive pairs q[0 .. nk) hosted on centre Z (host l = LH, other l = LO), then HRR / derivative / tile contraction
// into the lane's accumulator slots.
template <int LH, int LO, bool TR, bool PIPE, bool KT, int AUX, class Ring>
RIS_DEV void ris_phase(int nk, const double* __restrict__ q, double ZCx, double ZCy, double ZCz, double ZOx, double ZOy,
                       double ZOz, double alpha, double auxfac, const double* __restrict__ boys, Ring& ring, int nb,
                       const double* __restrict__ sc, double* __restrict__ slot)
{
    using K = RisClass<LH, LO>;
    constexpr int E = K::E;
    double acc[K::NACC];
#pragma unroll
    for (int i = 0; i < K::NACC; ++i) acc[i] = 0.0;
    if (PIPE && AUX == 0) {
        // front of primitive k+1 (record load, rsqrt(p + alpha), T: branch-free) next to Boys + recurrence of primitive k
        double2 r0 = *reinterpret_cast<const double2*>(q), r1 = *reinterpret_cast<const double2*>(q + 2);
        double2 r2 = *reinterpret_cast<const double2*>(q + 4), r3 = *reinterpret_cast<const double2*>(q + 6);
        RisPrimFront f;
        ris_prim_front(r0.x, r0.y, r1.x, r1.y, r3.y, ZCx, ZCy, ZCz, alpha, auxfac, f);
        for (int k = 0; k < nk; ++k) {
            const double* __restrict__ qn = q + (size_t)(k + 1 < nk ? k + 1 : k) * RIS_PRIM_FIELDS;
            const double2 n0 = *reinterpret_cast<const double2*>(qn), n1 = *reinterpret_cast<const double2*>(qn + 2);
            const double2 n2 = *reinterpret_cast<const double2*>(qn + 4), n3 = *reinterpret_cast<const double2*>(qn + 6);
            RisPrimFront fn;
            ris_prim_front(n0.x, n0.y, n1.x, n1.y, n3.y, ZCx, ZCy, ZCz, alpha, auxfac, fn);
            double F[E + 1];
            ris_boys<E>(f.T, boys, F, f.kappa);
            const double h2 = TR ? r3.x : r2.y, o2 = TR ? r2.y : r3.x;
            if constexpr (LO == 0) {
                const double hp = h2 * r2.x;
                ris_vrr<LH, LO>(F, r0.y, r1.x, r1.y, -f.q * f.X0, -f.q * f.X1, -f.q * f.X2, r2.x, f.q, h2, o2, acc, hp * ZOx, hp * ZOy,
                                hp * ZOz);
            } else {
                ris_vrr<LH, LO>(F, r0.y, r1.x, r1.y, -f.q * f.X0, -f.q * f.X1, -f.q * f.X2, r2.x, f.q, h2, o2, acc);
            }
            r0 = n0; r1 = n1; r2 = n2; r3 = n3; f = fn;
        }
    } else {
        for (int k = 0; k < nk; ++k, q += RIS_PRIM_FIELDS) {
            const double2 r0 = *reinterpret_cast<const double2*>(q);
            const double2 r1 = *reinterpret_cast<const double2*>(q + 2);
            const double2 r2 = *reinterpret_cast<const double2*>(q + 4);
            const double2 r3 = *reinterpret_cast<const double2*>(q + 6);
            if constexpr (AUX == 0)
                ris_prim_triplet<LH, LO>(r0.x, r0.y, r1.x, r1.y, r2.x, TR ? r3.x : r2.y, TR ? r2.y : r3.x, r3.y, ZCx, ZCy, ZCz,
                                         alpha, auxfac, boys, acc, ZOx, ZOy, ZOz);
            else
                ris_prim_triplet_p<LH, LO, AUX - 1>(r0.x, r0.y, r1.x, r1.y, r2.x, TR ? r3.x : r2.y, TR ? r2.y : r3.x, r3.y, ZCx, ZCy,
                                                    ZCz, alpha, auxfac, boys, acc, ZOx, ZOy, ZOz);
        }
    }
    ris_hrrc<LH, LO, TR, 33, KT ? 0 : 32>(acc, ZOx, ZOy, ZOz, ring, nb, sc, slot);
}

// KT: K-type contraction (Gamma^P tile, P-minor, one column per lane); else J-type (D tile shared by all lanes, scaled by
// c_aux[s][function]).  AUX: type of the auxiliary functions of this launch's list -- 0: s; 1, 2, 3: p_x, p_y, p_z (J only).
template <int LA, int LB, int PH, bool KT, int AUX = 0>
__global__ void __launch_bounds__(32 * RisGradTune<LA, LB>::NW, RisGradTune<LA, LB>::MINB) ris_grad_kernel(const RisGradParams prm)
{
    using Tune = RisGradTune<LA, LB>;
    constexpr int NEL = Tune::NEL;
    constexpr int NS = KT ? Tune::NSK : RIS_NB_MAX;          // upper bound of the ring; prm.ring_ns slots are in use
    extern __shared__ __align__(16) unsigned char sm_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const RisClassPack& pk = prm.pk;
    const int nb = prm.nb;
    const size_t wbytes = ris_grad_warp_smem(pk.task_prims, pk.kmax, nb, ris_grad_tile_doubles<LA, LB, KT>(prm.ring_ns));
    double* s_prim = reinterpret_cast<double*>(sm_raw + (size_t)warp * wbytes);
    RisPairRec* s_pair = reinterpret_cast<RisPairRec*>(s_prim + (size_t)RIS_PRIM_FIELDS * (pk.task_prims + pk.kmax));
    double* s_tile = reinterpret_cast<double*>(s_pair + pk.task_prims);      // tile ring (16-byte aligned)
    double* s_red = s_tile + ris_grad_tile_doubles<LA, LB, KT>(prm.ring_ns); // [6 nb][33]  pair side: A x,y,z, B x,y,z per state
    double* s_gaux = s_red + 6 * nb * 33;                                    // [3 nb][32]  aux side
    double* s_sc = s_gaux + 3 * nb * 32;                                     // [nb][32]    J: c_aux[s][P]
    const size_t gaux_off = (size_t)(reinterpret_cast<unsigned char*>(s_gaux) - (sm_raw + (size_t)warp * wbytes));

    // this lane's auxiliary function: position in the launch's list -> record (centre, exponent, N/alpha, atom, function index)
    const int pos = prm.p0 + blockIdx.y * 32 + lane;
    const bool live = pos < prm.p1;
    const int Pe = live ? pos : prm.p1 - 1;
    const double* ax = prm.aux + RIS_AUX_FIELDS * (size_t)Pe;
    const double Cx = ax[0], Cy = ax[1], Cz = ax[2], alpha = ax[3];
    const double auxfac = live ? ax[4] : 0.0;          // a dead lane computes exact zeros
    const int2 ids = *reinterpret_cast<const int2*>(ax + 5);
    const int P = ids.x;                               // the atom the function sits on: its gradient row
    if (!KT)
        for (int s = 0; s < nb; ++s) s_sc[s * 32 + lane] = prm.cscale[(size_t)s * prm.naux + ids.y];
    for (int i = 0; i < 6 * nb; ++i) s_red[i * 33 + lane] = 0.0;
    for (int i = 0; i < 3 * nb; ++i) s_gaux[i * 32 + lane] = 0.0;
    constexpr bool STAGED = !KT || Tune::STAGE_K;
    typename std::conditional<STAGED, RisTileRing<NEL, NS, KT>, RisTileDirectK>::type ring;
    if constexpr (STAGED) ring.buf = s_tile;
    ring.estride = (size_t)prm.estride; ring.sstride = (size_t)prm.sstride;
    ring.nb = nb; ring.ns = prm.ring_ns; ring.lane = lane;
    ring.nv = min(32, prm.p1 - prm.p0 - (int)blockIdx.y * 32);
    const double* __restrict__ tile_chunk = prm.tile + (KT ? (size_t)blockIdx.y * 32 : 0);
    int curA = -1, curB = -1;
    __syncwarp();

    // pair side: fixed-order sum over the lanes, one atomic per (state, centre, x); aux side keeps -(gA + gB)
    auto flush = [&]() {
        if (curA < 0) return;
        for (int s = 0; s < nb; ++s)
#pragma unroll
            for (int x = 0; x < 3; ++x)
                s_gaux[(s * 3 + x) * 32 + lane] -= s_red[(s * 6 + x) * 33 + lane] + s_red[(s * 6 + 3 + x) * 33 + lane];
        __syncwarp();
        if (lane < 6 * nb) {
            const double* r = s_red + lane * 33;
            double v = 0.0;
#pragma unroll 8
            for (int j = 0; j < 32; ++j) v += r[j];
            const int s = lane / 6, c = lane - 6 * s;
            const int at = c < 3 ? curA : curB;
            ris_grad_add(prm, ((size_t)s * prm.natoms + at) * 3 + (c < 3 ? c : c - 3), v);
        }
        __syncwarp();
        for (int i = 0; i < 6 * nb; ++i) s_red[i * 33 + lane] = 0.0;
        __syncwarp();
    };

    // Tasks are handed out by an atomic ticket counter per aux chunk; the ticket for the NEXT task is drawn before the
    // current one starts, so its latency is hidden.  Every warp ends within one task of the others, and a block that
    // becomes resident late finds the counter exhausted and leaves.
    int task = 0;
    if (lane == 0) task = atomicAdd(prm.task_ctr + blockIdx.y, 1);
    task = __shfl_sync(0xffffffffu, task, 0);
    while (task < pk.ntasks) {
        int next = 0;
        if (lane == 0) next = atomicAdd(prm.task_ctr + blockIdx.y, 1);
        const int ip0 = pk.task_begin[task], ip1 = pk.task_begin[task + 1];
        const long long q0 = pk.prim_off[ip0], q1 = pk.prim_off[ip1];
        __syncwarp();
        {   // stage the task: 16-byte copies, 4 per record
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
            if (pr.atA != curA || pr.atB != curB) { flush(); curA = pr.atA; curB = pr.atB; }
            const bool runA = PH != 2 && pr.nkA > 0, runB = LB > 0 && PH != 1 && pr.nkB > 0;
            ring.g = tile_chunk + ((size_t)pk.elem_off + (size_t)(ip0 + j) * NEL) * ring.estride;
            __syncwarp();                              // every lane is done with the previous pair's tile
            if (runA || runB) ring.begin();
            const double ACx = pr.Ax - Cx, ACy = pr.Ay - Cy, ACz = pr.Az - Cz;
            if (runA)
                ris_phase<LA, LB, false, Tune::PIPE, KT, AUX>(pr.nkA, q, ACx, ACy, ACz, pr.ABx, pr.ABy, pr.ABz, alpha, auxfac, prm.boys, ring,
                                                     nb, s_sc + lane, s_red + lane);
            q += (size_t)pr.nkA * RIS_PRIM_FIELDS;
            if constexpr (LB > 0) {        // (l,s) pairs are hosted on the l shell for every primitive pair: one phase
                if (runB) {
                    if (runA && !ring.holds_all()) { __syncwarp(); ring.begin(); }      // the ring has rolled past state 0
                    ris_phase<LB, LA, true, Tune::PIPE, KT, AUX>(pr.nkB, q, ACx - pr.ABx, ACy - pr.ABy, ACz - pr.ABz, -pr.ABx, -pr.ABy,
                                                            -pr.ABz, alpha, auxfac, prm.boys, ring, nb, s_sc + lane, s_red + lane);
                }
            }
            q += (size_t)pr.nkB * RIS_PRIM_FIELDS;
        }
        if (prm.det != nullptr) {
            // deterministic mode: which warp runs which task varies from run to run, so every task hands over its own
            // sums (integer atomics: exact, order-independent) instead of carrying FP64 partial sums into the next task
            flush();
            curA = curB = -1;
            if (live)
                for (int i = 0; i < 3 * nb; ++i) {
                    ris_grad_add(prm, ((size_t)(i / 3) * prm.natoms + P) * 3 + (i % 3), s_gaux[i * 32 + lane]);
                    s_gaux[i * 32 + lane] = 0.0;
                }
        }
        task = __shfl_sync(0xffffffffu, next, 0);
    }
    flush();

    // aux side: the warps of the block hold the same 32 aux functions
    __syncthreads();
    if (warp == 0 && live) {
        for (int i = 0; i < 3 * nb; ++i) {
            double v = 0.0;
#pragma unroll
            for (int w = 0; w < Tune::NW; ++w)
                v += reinterpret_cast<const double*>(sm_raw + (size_t)w * wbytes + gaux_off)[i * 32 + lane];
            const int s = i / 3, x = i - 3 * s;
            ris_grad_add(prm, ((size_t)s * prm.natoms + P) * 3 + x, v);
        }
    }
}

template <int LA, int LB, int PH, bool KT, int AUX>
cudaError_t ris_launch_grad_phase(const RisGradParams& p0_, cudaStream_t st)
{
    // ring slots: all states when they fit the class budget, fewer when the task records of a long contraction (kmax up
    // to 576 primitive pairs) leave less than that of the 227 KB a block may use
    RisGradParams p = p0_;
    constexpr int NSMAX = KT ? RisGradTune<LA, LB>::NSK : RIS_NB_MAX;
    constexpr int NW = RisGradTune<LA, LB>::NW;
    auto smem_of = [&](int ns) { return NW * ris_grad_warp_smem(p.pk.task_prims, p.pk.kmax, p.nb, ris_grad_tile_doubles<LA, LB, KT>(ns)); };
    auto resident_of = [&](size_t bytes) {
        return std::max(1, std::min<int>(RisGradTune<LA, LB>::MINB * RIS_GRAD_WARPS / NW, (int)((227 * 1024) / (bytes + 1024))));
    };
    // A slot per state (the fast path of the ring) when that costs no resident block; otherwise the smallest ring (K: one or
    // two slots, refilled state by state) -- a half-sized ring gives neither.
    const int ns_full = p.nb < NSMAX ? p.nb : NSMAX;
    const int ns_lo = KT ? std::min(p.nb, RisGradTune<LA, LB>::NSK_LO) : ns_full;
    p.ring_ns = (smem_of(ns_full) <= (size_t)227 * 1024 && resident_of(smem_of(ns_full)) >= resident_of(smem_of(ns_lo))) ? ns_full : ns_lo;
    size_t smem = 0;
    for (;; --p.ring_ns) {
        smem = smem_of(p.ring_ns);
        if (smem <= 227 * 1024 || p.ring_ns == 1) break;
    }
    // the opt-in is per device and context: set it at every launch that needs it (a host-side call of ~1 us) instead of
    // caching it in process-wide state
    if (smem > 48 * 1024) {
        const cudaError_t e = cudaFuncSetAttribute(ris_grad_kernel<LA, LB, PH, KT, AUX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    // blockIdx.y: chunks of 32 aux functions; blockIdx.x: the blocks of a chunk, together one resident wave of
    // long-lived warps drawing tasks (few aux-side atomics, no wave quantisation)
    const int ny = (p.p1 - p.p0 + 31) / 32;
    const int nbt = (p.pk.ntasks + NW - 1) / NW;
    // resident blocks per SM: the register target, or what the shared memory of the block allows
    const int resident = resident_of(smem);
    const int nx = std::max(1, std::min(nbt, (p.nsm * resident + ny - 1) / ny));
    ris_grad_kernel<LA, LB, PH, KT, AUX><<<dim3(nx, ny), 32 * NW, smem, st>>>(p);
    return cudaGetLastError();
}

// p.task_ctr holds two zeroed ticket arrays of ny counters each (one per phase launch)
template <int LA, int LB, bool KT, int AUX>
cudaError_t ris_launch_grad_t(const RisGradParams& p, cudaStream_t st)
{
    if constexpr (RisGradTune<LA, LB>::SPLIT) {
        RisGradParams q = p;
        cudaError_t e = ris_launch_grad_phase<LA, LB, 1, KT, AUX>(q, st);
        if (e != cudaSuccess) return e;
        q.task_ctr = p.task_ctr + (p.p1 - p.p0 + 31) / 32;
        return ris_launch_grad_phase<LA, LB, 2, KT, AUX>(q, p.phase2_stream ? p.phase2_stream : st);
    } else {
        return ris_launch_grad_phase<LA, LB, 0, KT, AUX>(p, st);
    }
}

// p.lstride selects the contraction type (K: P-minor tile), p.aux_type the auxiliary function type of the list (J only)
template <int LA, int LB>
cudaError_t ris_launch_grad(const RisGradParams& p, cudaStream_t st)
{
    if (p.pk.npairs <= 0 || p.pk.ntasks <= 0 || p.p1 <= p.p0) return cudaSuccess;
    if (p.lstride) return p.aux_type == 0 ? ris_launch_grad_t<LA, LB, true, 0>(p, st) : cudaErrorInvalidValue;
    switch (p.aux_type) {
    case 0: return ris_launch_grad_t<LA, LB, false, 0>(p, st);
    case 1: return ris_launch_grad_t<LA, LB, false, 1>(p, st);
    case 2: return ris_launch_grad_t<LA, LB, false, 2>(p, st);
    case 3: return ris_launch_grad_t<LA, LB, false, 3>(p, st);
    default: return cudaErrorInvalidValue;
    }
}
