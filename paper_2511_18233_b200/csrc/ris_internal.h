// ris_internal.h -- structures shared between the translation units of libris_b200.so.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

constexpr int RIS_LMAX = 3;
constexpr int RIS_NCLASS = 10;          // (la,lb), la >= lb, la <= 3
constexpr int RIS_AUX_FIELDS = 8;       // doubles per aux record (RisGradParams::aux)
constexpr int RIS_PRIM_FIELDS = 8;      // p, (P-Z)x, (P-Z)y, (P-Z)z, 1/(2p), 2a, 2b, coef   (Z = host centre); one 64-byte record
constexpr int RIS_GRAD_WARPS = 4;       // warps per class-kernel block
constexpr int RIS_GRAD_THREADS = 32 * RIS_GRAD_WARPS;
constexpr int RIS_TASK_PRIMS = 32;      // a warp task = the shell pairs whose first primitive pair falls in one window of
                                        // ris_task_prims(class) <= RIS_TASK_PRIMS packed primitive pairs (so a task holds
                                        // fewer than window + kmax of them)
constexpr int RIS_NB_MAX = 5;           // states per class-kernel launch (per-state gradient slots in shared memory)

__host__ __device__ constexpr int ris_class_id(int la, int lb) { return la * (la + 1) / 2 + lb; }
__host__ __device__ constexpr int ris_ncart(int l) { return (l + 1) * (l + 2) / 2; }
// task window by class weight: a (d,d) primitive triplet costs ~10x an (s,s) one, and a task should stay ~10-20 us
__host__ __device__ constexpr int ris_task_prims(int la, int lb) { return la + lb <= 1 ? 24 : (la + lb <= 2 ? 32 : (la + lb <= 3 ? 16 : 8)); }

// One packed shell pair (64 bytes, read by a whole warp as a broadcast).
struct __align__(16) RisPairRec {
    double Ax, Ay, Az;       // centre of mu
    double ABx, ABy, ABz;    // A - B
    int atA, atB;            // atom of mu, atom of nu
    int nkA, nkB;            // surviving primitive pairs hosted on A (a >= b; stored first) / on B (b > a)
};
static_assert(sizeof(RisPairRec) == 64, "pair record layout");

// Packed shell pairs of one class (device pointers).  The pairs are sorted by (atom of mu, atom of nu), so that the
// class kernel keeps the pair-side gradient of an atom pair in registers across its shell pairs.
struct RisClassPack {
    int la, lb;
    int npairs;            // surviving shell pairs
    int kmax;              // max surviving primitive pairs per shell pair
    long long nprim;       // surviving primitive pairs in the class
    int ntasks;            // warp tasks (windows of task_prims primitive pairs)
    int task_prims;
    RisPairRec* pairs;     // [npairs]
    int* ao;               // [2][npairs]  first AO of mu, first AO of nu
    float* symf;           // [npairs]     1 (mu != nu shell) or 0.5 (same shell): folds D + D^T onto unique pairs
    long long* prim_off;   // [npairs + 1] first primitive-pair record of the pair (exclusive scan)
    double* prim;          // [nprim][8]
    int* task_begin;       // [ntasks + 1] first pair of the task
    long long elem_off;    // first packed Cartesian pair element of the class; pair ip holds elements
                           // elem_off + ip * nca * ncb + (ca * ncb + cb)
};

// Launch description of one class kernel (by value to the kernel).
struct RisGradParams {
    RisClassPack pk;
    int naux, natoms;        // naux: functions in the coefficient vector (row length of cscale / v)
    int nsm;                 // SMs of the context's device (grid sizing)
    // aux records of this launch's LIST of auxiliary functions, 8 doubles each: Cx, Cy, Cz, alpha, N/alpha, then two ints
    // (atom of the function -> gradient row, index of the function -> column of cscale / v), one double of padding.
    // K type and the default J set: the list is all naux s functions (atom = index).  A J-fit set with p functions (NEXT-2)
    // is run as four lists -- s, p_x, p_y, p_z -- with aux_type 0..3 selecting the kernel specialisation.
    const double* aux;
    int aux_type;
    const double* boys;      // table for M = E of this class
    // packed tiles: element el of state s for aux P sits at tile[s*sstride + el*estride + (P - p0)*lstride]
    //   J: estride 1, lstride 0 (D tile, the same for every P);  K: estride = padded P-batch, lstride 1 (Gamma^P)
    const double* tile;
    long long sstride, estride;
    int lstride;
    const double* cscale;    // J: c_aux[nb][naux]; K: nullptr
    int nb;
    int ring_ns;             // slots of the shared-memory tile ring (set by the launcher)
    int p0, p1;              // range of list positions of this launch; blockIdx.y selects 32 of them, one per lane
    int* task_ctr;           // [chunks of 32 aux] zeroed ticket counters of this launch (dynamic task hand-out)
    double* grad;            // [nb][natoms][3], accumulated with atomics
    unsigned long long* det; // deterministic mode: [nb][natoms][3][2] fixed-point accumulators (hi, lo), else nullptr
    int* det_flag;           // set to 1 when a contribution leaves the fixed-point range
    cudaStream_t phase2_stream;   // host side only: when set, the second host-phase launch of a split class goes here
                                  // (small molecules: the two phases run side by side); nullptr = the launch stream
};

// Deterministic reduction (ris_options.deterministic): a contribution x is added as the integer pair
//   hi = floor(x 2^28),  lo = floor((x 2^28 - hi) 2^32)        value = hi 2^-28 + lo 2^-60
// with two 64-bit INTEGER atomics; integer addition is associative, so the result does not depend on the order in
// which warps arrive (resolution 2^-60 ~ 8.7e-19 per contribution, range |x| < 2^34, |sum| < 2^35).
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

typedef cudaError_t (*ris_grad_launcher)(const RisGradParams&, cudaStream_t);
extern ris_grad_launcher ris_grad_launchers[RIS_NCLASS];


// ---- per-class configuration of the class kernels, shared by host sizing code and the kernel templates ----------------
// the heavy classes (l_mu + l_nu >= RIS_SPLIT_L) run their two host-centre phases as two launches (ris_grad_kernel.cuh)
#ifndef RIS_SPLIT_L
#define RIS_SPLIT_L 4
#endif
__host__ __device__ constexpr bool ris_grad_split(int la, int lb) { return la + lb >= RIS_SPLIT_L; }
// K tiles of the biggest classes (60 / 100 elements: 15-26 KB per state and warp) are read straight from global memory
__host__ __device__ constexpr bool ris_grad_stage_k(int la, int lb) { return ris_ncart(la) * ris_ncart(lb) < 60; }

// Dynamic shared memory of one warp of a class-kernel block with a tile ring of `tile_doubles` (host + device agree
// through this; ris_grad_kernel.cuh).
__host__ __device__ inline size_t ris_grad_warp_smem(int window, int kmax, int nb, int tile_doubles)
{
    return (size_t)64 * (window + kmax)              // primitive-pair records of the task (window = pk.task_prims)
         + (size_t)64 * window                       // pair records of the task
         + (size_t)8 * (6 * nb * 33 + 3 * nb * 32 + nb * 32)   // pair-side slots [6 nb][33], aux-side slots, scales
         + (size_t)8 * tile_doubles;                 // tile ring
}
// Largest number of states per launch (<= RIS_NB_MAX) with which a block of class (la,lb) and its smallest tile ring (one
// slot) stays within the 227 KB a block may use; 0 if not even one state fits.
inline int ris_grad_nb_cap(int la, int lb, int kmax, bool ktype)
{
    const int nel = ris_ncart(la) * ris_ncart(lb);
    const int ring = ktype ? (ris_grad_stage_k(la, lb) ? nel * 32 : 0) : ((nel + 1) & ~1);
    for (int nb = RIS_NB_MAX; nb >= 1; --nb)
        if (RIS_GRAD_WARPS * ris_grad_warp_smem(ris_task_prims(la, lb), kmax, nb, ring) <= (size_t)227 * 1024)
            return nb;
    return 0;
}
