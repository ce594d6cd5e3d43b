// ris_api.cu -- C ABI (include/ris.h), context, host-side orchestration, and the small kernels:
// tile packing, two-centre term (S5), FP64 probe.  The class kernels live in ris_grad_kernel.cuh
// (one translation unit per class under generated/), the Gamma^P GEMMs in ris_gemm.cuh.
#include "../../include/ris.h"
#include "../../include/ris_bench.h"
#include "ris_boys_table.h"
#include "ris_core.cuh"
#include "ris_gemm.cuh"
#include "ris_internal.h"
#include "ris_setup.cuh"
#include "ris_sph.cuh"

constexpr int RIS_NPRIM_MAX = 24;        // primitives per shell (kmax <= 576: the class-kernel task fits in shared memory)

#include <algorithm>
#include <utility>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

// --------------------------------------------------------------------------------------- errors
static thread_local std::string g_cuda_err = "no CUDA error recorded";

static int cuda_fail(cudaError_t e, const char* what, int line)
{
    char buf[512];
    snprintf(buf, sizeof buf, "CUDA error at %s (ris_api.cu:%d): %s", what, line, cudaGetErrorString(e));
    g_cuda_err = buf;
    return RIS_ECUDA;
}
#define CU(x) do { cudaError_t e__ = (x); if (e__ != cudaSuccess) return cuda_fail(e__, #x, __LINE__); } while (0)

extern "C" const char* ris_strerror(int status)
{
    switch (status) {
    case RIS_OK: return "success";
    case RIS_EINVAL: return "invalid argument";
    case RIS_ENOMEM: return "out of memory";
    case RIS_ECUDA: return g_cuda_err.c_str();
    default: return "unknown status";
    }
}

// --------------------------------------------------------------------------------------- context
struct ProfRec { const char* name; cudaEvent_t e0, e1; double flops, bytes; };

// Stored MO-basis tensors and scratch of the coupling-matrix products (ris_resp.cuh)
struct RisResp {
    bool ready = false;
    int no = 0, nv = 0, nop = 0, nvp = 0;      // nocc, nvir and their even paddings
    int nz = 0, pc = 0, nKp = 0;               // split of the (P, j) contraction: nz ranges of pc aux functions, nKp = nz pc
    double *TJ = nullptr, *Tvv = nullptr, *BooT = nullptr, *Bov = nullptr, *TovT = nullptr;
    double *Xp = nullptr, *Y = nullptr, *part = nullptr, *uw = nullptr;
    int vc = 0, nchunk = 0;                    // vectors per pass the scratch is sized for; chunks of the Coulomb reduction
};

struct ris_ctx {
    int device = 0;
    int nsm = 0;                       // SMs of `device` (grid sizing of the class kernels)
    cudaStream_t stream = nullptr;
    ris_options opt{};
    int natoms = 0, nshells = 0, nao = 0, naux = 0;   // nao: Cartesian AOs (what the kernels run on)
    int nao_in = 0;                    // AOs of the caller's basis: nao, or sum (2l+1) with opt.spherical (ris_sph.cuh)
    int *d_sph0 = nullptr, *d_sph_lc = nullptr;   // spherical mode: per Cartesian AO the first spherical AO of its shell, 16 l + component
    double* d_coords = nullptr;
    double* d_aux = nullptr;           // [naux][RIS_AUX_FIELDS] the default set: one s function per atom (K type; J type too
                                       // unless ris_set_jfit gave the J term a set of its own)
    // J-fit set (NEXT-2): s and p functions.  Without ris_set_jfit these alias the default set.
    bool jfit = false;
    int naux_J = 0;                    // functions of the J-fit set
    double* d_jfn = nullptr;           // [naux_J][RIS_AUX_FIELDS] records in FUNCTION order (two-centre kernels)
    double* d_jlist[4] = {nullptr};    // the same records grouped by type: s, p_x, p_y, p_z (class kernels: one launch each)
    int jcnt[4] = {0, 0, 0, 0};
    std::vector<int> h_jlist_fn[4];    // function index of every list entry (ascending): ranges of functions -> list positions
    int *d_atom_fn_off = nullptr, *d_atom_fn = nullptr;   // CSR atom -> functions of the J-fit set
    double* d_chol_J = nullptr;        // Cholesky factor of the J-fit metric (explicit set only; else d_chol)
    int *d_shell_atom = nullptr, *d_shell_l = nullptr, *d_shell_nprim = nullptr, *d_shell_poff = nullptr, *d_shell_ao = nullptr;
    double *d_pexp = nullptr, *d_pcoef = nullptr;
    RisClassPack cls[RIS_NCLASS]{};
    std::vector<void*> owned;          // every device allocation of the packed data
    std::vector<double> h_coords;      // host copy of the geometry (ris_set_jfit places its functions on the atoms)
    long long nelem_real = 0, npairs_total = 0, nprim_surv = 0, nprim_total = 0;
    double* d_boys[9] = {nullptr};     // Boys tables of top order M = 0..8 (M = 8: d/dR of (ff|p))
    double* d_minv = nullptr;          // [naux][nauxp] inverse metric (built by the first ris_fit_K)
    double* d_minv_J = nullptr;        // the same for an explicit J-fit set
    // band of the spatially ordered AO index per 64-row block (from the GEMM-2 block list): columns
    // [rb_jlo*64, (rb_jlo*64 + rb_kw)) hold every surviving partner of the block's rows
    std::vector<int> rb_jlo, rb_kw;
    std::vector<long long> rb_off;     // offset (doubles) of the block's [64][rb_kw] slab within one P
    long long slab_stride = 0;
    int *d_rb_jlo = nullptr, *d_rb_kw = nullptr;
    long long* d_rb_off = nullptr;
    double* d_chol = nullptr;          // [naux][naux] lower Cholesky factor of the aux metric (built by the first ris_fit_J)
    // Gamma^P GEMM-2 (ris_gemm.cuh, scatter mode): per AO position nu' the gathered list of its surviving partners
    int* d_ao_pos = nullptr;           // [nao] spatial position of AO
    int* d_ao_order = nullptr;         // [nao] AO at spatial position
    int nblk = 0;                      // 64-row blocks of the spatial AO order (fit_K bands)
    int ntiles = 0;                    // GEMM-2 tiles: RIS_G2_BM partner rows of one column problem each
    long long g2_entries = 0;          // partner-list entries (2 per packed pair element)
    int2* d_g2tiles = nullptr;         // [ntiles] (column problem nu', first entry of the tile in d_g2rows / d_g2code)
    int* d_g2rows = nullptr;           // [ntiles * RIS_G2_BM] partner position mu' (A row), -1 = padding
    int* d_g2code = nullptr;           // [ntiles * RIS_G2_BM] packed element << 1 | (symmetry factor 1/2), -1 = padding
    // grow-only scratch
    cudaStream_t copy_stream = nullptr;           // *_host entry points: H2D of B, one state ahead of the GEMMs
    std::vector<cudaEvent_t> copy_ev;             // [state] B of that state has landed
    cudaStream_t side[RIS_NCLASS] = {nullptr};    // class kernels of small molecules run concurrently on these
    // Small molecules (the class kernels run side by side, see launch_classes): a device-pointer call whose arguments repeat
    // is captured into a CUDA graph the second time and replayed from then on (run_graphed).
    struct GraphSlot { std::vector<unsigned long long> key; cudaGraphExec_t exec = nullptr; };
    GraphSlot gslot[2];                           // ris_grad_J(_range), ris_grad_K(_range)
    cudaStream_t cap_stream = nullptr;            // the capture runs on a stream of our own (the caller's may be the legacy
                                                  // default stream, which cannot be captured); the graph is launched into the caller's
    bool small = false;                           // set by ris_setup: no class fills the GPU with its one resident wave
    cudaStream_t side2[RIS_NCLASS] = {nullptr};   // ... and the second host-phase launch of a split (heavy) class on these
    cudaEvent_t join2_ev[RIS_NCLASS] = {nullptr};
    cudaEvent_t join_ev[RIS_NCLASS] = {nullptr}, fork_ev = nullptr;
    cudaEvent_t copy_extra = nullptr;             // the extra payload of upload_B_chunked has landed
    cudaEvent_t copy_gate = nullptr;              // compute stream -> copy stream: the staging buffer is free
    void* ws[32] = {nullptr};
    size_t ws_bytes[32] = {0};
    RisResp resp;
    int last_pbatch = 0;
    std::vector<ProfRec> prof;
    std::vector<cudaEvent_t> ev_pool;
};

enum { WS_TILE = 0, WS_H = 1, WS_UNUSED2 = 2, WS_IN0 = 3, WS_IN1 = 4, WS_IN2 = 5, WS_OUT = 6, WS_COCC = 7, WS_DET = 8, WS_CTR = 9,
       WS_FIT_I = 10, WS_FIT_SLAB = 11, WS_FIT_UT = 12, WS_FIT_T = 13, WS_FIT_TT = 14, WS_FIT_CV = 15, WS_FIT_CO = 16, WS_HC = 17, WS_HDQ = 18, WS_HD = 19, WS_RESP_T = 20, WS_RESP_B = 21, WS_SPH_A = 22, WS_SPH_B = 23, WS_N = 24 };
static_assert(WS_N <= 32, "ris_ctx::ws holds 32 workspace slots");

// The captured graphs hold workspace and list pointers: drop them whenever one of those may have changed.
static void graphs_invalidate(ris_ctx* c)
{
    for (auto& g : c->gslot) {
        if (g.exec) cudaGraphExecDestroy(g.exec);
        g.exec = nullptr;
        g.key.clear();
    }
}

static int ws_get(ris_ctx* c, int slot, size_t bytes, void** out)
{
    if (c->ws_bytes[slot] < bytes) {
        graphs_invalidate(c);
        if (c->ws[slot]) { CU(cudaStreamSynchronize(c->stream)); CU(cudaFree(c->ws[slot])); c->ws[slot] = nullptr; c->ws_bytes[slot] = 0; }
        cudaError_t e = cudaMalloc(&c->ws[slot], bytes);
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return RIS_ENOMEM; }
        CU(e);
        c->ws_bytes[slot] = bytes;
    }
    *out = c->ws[slot];
    return RIS_OK;
}

template <class T> static int dev_alloc(ris_ctx* c, T** p, size_t n, bool zero)
{
    // stream-ordered allocation from the device's default memory pool: a context built after another one was destroyed
    // (a new geometry in a running process) gets its ~50 buffers back from the pool instead of from the driver
    void* q = nullptr;
    cudaError_t e = cudaMallocAsync(&q, std::max<size_t>(n, 1) * sizeof(T), c->stream);
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return RIS_ENOMEM; }
    CU(e);
    c->owned.push_back(q);
    if (zero) CU(cudaMemsetAsync(q, 0, std::max<size_t>(n, 1) * sizeof(T), c->stream));
    *p = (T*)q;
    return RIS_OK;
}

template <class T> static int dev_upload(ris_ctx* c, T** p, const T* h, size_t n)
{
    int rc = dev_alloc(c, p, n, false);
    if (rc) return rc;
    if (n) CU(cudaMemcpyAsync(*p, h, n * sizeof(T), cudaMemcpyHostToDevice, c->stream));
    return RIS_OK;
}

// profiling: events around a launch when opt.profile is set
struct ProfScope {
    ris_ctx* c; int idx = -1; cudaStream_t st;
    // flops / bytes: ALGORITHMIC work of the launch; st: the stream the launch
    // goes to when it is not the context's own (concurrent class kernels of small molecules)
    ProfScope(ris_ctx* c_, const char* name, double flops = 0.0, double bytes = 0.0, cudaStream_t st_ = nullptr, bool own = true)
        : c(c_), st(own ? c_->stream : st_)
    {
        if (!c->opt.profile) return;
        ProfRec r; r.name = name; r.flops = flops; r.bytes = bytes;
        if (cudaEventCreate(&r.e0) != cudaSuccess || cudaEventCreate(&r.e1) != cudaSuccess) return;
        cudaEventRecord(r.e0, st);
        c->prof.push_back(r);
        idx = (int)c->prof.size() - 1;
    }
    ~ProfScope() { if (idx >= 0) cudaEventRecord(c->prof[idx].e1, st); }
};

extern "C" int ris_profile_reset(ris_ctx* c)
{
    if (!c) return RIS_EINVAL;
    for (auto& r : c->prof) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
    c->prof.clear();
    return RIS_OK;
}
extern "C" int ris_profile_count(ris_ctx* c) { return c ? (int)c->prof.size() : RIS_EINVAL; }
extern "C" int ris_profile_get(ris_ctx* c, int i, const char** name, float* ms)
{
    if (!c || i < 0 || i >= (int)c->prof.size()) return RIS_EINVAL;
    CU(cudaEventSynchronize(c->prof[i].e1));
    CU(cudaEventElapsedTime(ms, c->prof[i].e0, c->prof[i].e1));
    *name = c->prof[i].name;
    return RIS_OK;
}

extern "C" int ris_profile_enable(ris_ctx* c, int on)
{
    if (!c) return RIS_EINVAL;
    c->opt.profile = on ? 1 : 0;
    return RIS_OK;
}

extern "C" int ris_profile_get_work(ris_ctx* c, int i, double* flops, double* bytes)
{
    if (!c || i < 0 || i >= (int)c->prof.size() || !flops || !bytes) return RIS_EINVAL;
    *flops = c->prof[i].flops;
    *bytes = c->prof[i].bytes;
    return RIS_OK;
}

// --------------------------------------------------------------------------------------- class launchers
#define DECL(la, lb) cudaError_t ris_launch_grad_##la##lb(const RisGradParams&, cudaStream_t);
DECL(0, 0) DECL(1, 0) DECL(1, 1) DECL(2, 0) DECL(2, 1) DECL(2, 2) DECL(3, 0) DECL(3, 1) DECL(3, 2) DECL(3, 3)
#undef DECL
ris_grad_launcher ris_grad_launchers[RIS_NCLASS] = {
    ris_launch_grad_00, ris_launch_grad_10, ris_launch_grad_11, ris_launch_grad_20, ris_launch_grad_21,
    ris_launch_grad_22, ris_launch_grad_30, ris_launch_grad_31, ris_launch_grad_32, ris_launch_grad_33};
#define DECL(la, lb) cudaError_t ris_launch_int_##la##lb(const RisGradParams&, cudaStream_t);
DECL(0, 0) DECL(1, 0) DECL(1, 1) DECL(2, 0) DECL(2, 1) DECL(2, 2) DECL(3, 0) DECL(3, 1) DECL(3, 2) DECL(3, 3)
#undef DECL
static const ris_grad_launcher ris_int_launchers[RIS_NCLASS] = {
    ris_launch_int_00, ris_launch_int_10, ris_launch_int_11, ris_launch_int_20, ris_launch_int_21,
    ris_launch_int_22, ris_launch_int_30, ris_launch_int_31, ris_launch_int_32, ris_launch_int_33};
#define DECL(la, lb) cudaError_t ris_launch_ints_##la##lb(const RisGradParams&, cudaStream_t);
DECL(0, 0) DECL(1, 0) DECL(1, 1) DECL(2, 0) DECL(2, 1) DECL(2, 2) DECL(3, 0) DECL(3, 1) DECL(3, 2) DECL(3, 3)
#undef DECL
static const ris_grad_launcher ris_ints_launchers[RIS_NCLASS] = {
    ris_launch_ints_00, ris_launch_ints_10, ris_launch_ints_11, ris_launch_ints_20, ris_launch_ints_21,
    ris_launch_ints_22, ris_launch_ints_30, ris_launch_ints_31, ris_launch_ints_32, ris_launch_ints_33};
static const char* const kIntNames[RIS_NCLASS] = {
    "ris_int_kernel<0,0>", "ris_int_kernel<1,0>", "ris_int_kernel<1,1>", "ris_int_kernel<2,0>", "ris_int_kernel<2,1>",
    "ris_int_kernel<2,2>", "ris_int_kernel<3,0>", "ris_int_kernel<3,1>", "ris_int_kernel<3,2>", "ris_int_kernel<3,3>"};
static const char* const kGradNames[RIS_NCLASS] = {
    "ris_grad_kernel<0,0>", "ris_grad_kernel<1,0>", "ris_grad_kernel<1,1>", "ris_grad_kernel<2,0>", "ris_grad_kernel<2,1>",
    "ris_grad_kernel<2,2>", "ris_grad_kernel<3,0>", "ris_grad_kernel<3,1>", "ris_grad_kernel<3,2>", "ris_grad_kernel<3,3>"};
// Algorithmic FP64 flops per primitive triplet by E = la + lb + 1 (SURVEY.md 8(d) model: setup ~45, Boys ~30 + 4E,
// 7 flops per OS-VRR intermediate, scaled accumulation), plus 12 nca ncb flops per contracted triplet and state.
static const double kModelFlopsByE[9] = {90.0, 140.0, 250.0, 450.0, 750.0, 1250.0, 2000.0, 3100.0, 4600.0};
// heaviest class first (flops per primitive triplet), so the tail is made of light kernels
static const int kClassOrder[RIS_NCLASS] = {9, 8, 7, 5, 6, 4, 3, 2, 1, 0};

// --------------------------------------------------------------------------------------- setup
// GEMM-2 partner lists.  Every packed pair element e = (mu, nu) with symmetry factor f emits two entries:
//   into the list of column nu':  (row mu', e, f)   -- adds f Gamma^P_{mu nu} to tile[e][P]
//   into the list of column mu':  (row nu', e, f)   -- adds f Gamma^P_{nu mu}
// (a same-shell pair holds (ca,cb) and (cb,ca) as elements of their own, each with f = 1/2; its diagonal elements get
// two entries of 1/2 Gamma_{mu mu}).  Pass 1 counts per column and records, per 64-row block of the spatial AO order,
// the range of partner blocks (the bands of ris_fit_K).
__global__ void ris_k_g2_count(RisClassPack pk, const int* __restrict__ ao_pos, int* __restrict__ cnt, volatile int* jlo,
                               volatile int* jhi)
{
    const int nel = ris_ncart(pk.la) * ris_ncart(pk.lb), ncb = ris_ncart(pk.lb);
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)pk.npairs * nel) return;
    const int ip = (int)(idx / nel), e = (int)(idx - (long long)ip * nel), ca = e / ncb, cb = e - ca * ncb;
    const int r = ao_pos[pk.ao[ip]] + ca, q = ao_pos[pk.ao[(size_t)pk.npairs + ip]] + cb;
    atomicAdd(&cnt[q], 1);
    atomicAdd(&cnt[r], 1);
    const int I = r / RIS_GTILE2, J = q / RIS_GTILE2;
    // (read first: after the first few elements of a block pair nothing changes any more, and ~50 addresses would
    // otherwise serialise a million atomics)
    if (J < jlo[I]) atomicMin((int*)&jlo[I], J);
    if (J > jhi[I]) atomicMax((int*)&jhi[I], J);
    if (I < jlo[J]) atomicMin((int*)&jlo[J], I);
    if (I > jhi[J]) atomicMax((int*)&jhi[J], I);
}

// One block: tiles per column = ceil(cnt / BM); tbase[nu] = exclusive scan; tbase[nao] = total.
__global__ void __launch_bounds__(1024) ris_k_g2_scan(int nao, int bm, const int* __restrict__ cnt, int* __restrict__ tbase)
{
    __shared__ int part[1024];
    const int t = threadIdx.x, per = (nao + 1023) / 1024;
    const int i0 = min(t * per, nao), i1 = min(i0 + per, nao);
    int sum = 0;
    for (int i = i0; i < i1; ++i) sum += (cnt[i] + bm - 1) / bm;
    part[t] = sum;
    __syncthreads();
    if (t == 0) {
        int run = 0;
        for (int k = 0; k < 1024; ++k) { const int v = part[k]; part[k] = run; run += v; }
        tbase[nao] = run;
    }
    __syncthreads();
    int run = part[t];
    for (int i = i0; i < i1; ++i) { tbase[i] = run; run += (cnt[i] + bm - 1) / bm; }
}

__global__ void ris_k_g2_fill(RisClassPack pk, const int* __restrict__ ao_pos, int bm, const int* __restrict__ tbase,
                              int* __restrict__ fillctr, int* __restrict__ rows, int* __restrict__ code)
{
    const int nel = ris_ncart(pk.la) * ris_ncart(pk.lb), ncb = ris_ncart(pk.lb);
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)pk.npairs * nel) return;
    const int ip = (int)(idx / nel), e = (int)(idx - (long long)ip * nel), ca = e / ncb, cb = e - ca * ncb;
    const int r = ao_pos[pk.ao[ip]] + ca, q = ao_pos[pk.ao[(size_t)pk.npairs + ip]] + cb;
    const int c = (int)(((pk.elem_off + idx) << 1) | (pk.symf[ip] < 0.75f ? 1 : 0));
    int k = atomicAdd(&fillctr[q], 1);
    rows[(size_t)tbase[q] * bm + k] = r; code[(size_t)tbase[q] * bm + k] = c;
    k = atomicAdd(&fillctr[r], 1);
    rows[(size_t)tbase[r] * bm + k] = q; code[(size_t)tbase[r] * bm + k] = c;
}

__global__ void ris_k_g2_tiles(int nao, int bm, const int* __restrict__ tbase, int2* __restrict__ tiles)
{
    const int nu = blockIdx.x * blockDim.x + threadIdx.x;
    if (nu >= nao) return;
    for (int t = tbase[nu]; t < tbase[nu + 1]; ++t) tiles[t] = make_int2(nu, t * bm);
}

// Morton (Z-order) code of a point on a 3-bohr grid: the spatial AO order that keeps the surviving pairs of an
// extended molecule in a narrow band of blocks.
static unsigned long long morton3(const double* r, const double* lo)
{
    unsigned long long code = 0;
    for (int d = 0; d < 3; ++d) {
        const unsigned long long q = (unsigned long long)std::max(0.0, std::floor((r[d] - lo[d]) / 3.0));
        for (int b = 0; b < 20; ++b) code |= ((q >> b) & 1ull) << (3 * b + d);
    }
    return code;
}

// One auxiliary-function record: centre, exponent, N/alpha, then (atom, function index), (l, component) as int pairs.
//   s: N = (2 alpha/pi)^(3/4);   p_i: N (r - C)_i exp(-alpha |r-C|^2) with N = (2 alpha/pi)^(3/4) 2 sqrt(alpha)
static void aux_record(double* r, const double* xyz, double al, int l, int comp, int atom, int fn)
{
    const double N = std::pow(2.0 * al / M_PI, 0.75) * (l == 1 ? 2.0 * std::sqrt(al) : 1.0);
    r[0] = xyz[0]; r[1] = xyz[1]; r[2] = xyz[2]; r[3] = al; r[4] = N / al;
    const int ids[4] = {atom, fn, l, comp};
    std::memcpy(r + 5, ids, sizeof ids);
    r[7] = 0.0;
}

extern "C" int ris_setup(ris_ctx** out, int natoms, const double* coords, int nshells, const int32_t* shell_atom,
                         const int32_t* shell_l, const int32_t* shell_nprim, const int32_t* shell_prim_off,
                         const double* prim_exp, const double* prim_coef, const double* aux_exponents,
                         const ris_options* opt, void* cuda_stream)
{
    if (!out) return RIS_EINVAL;
    *out = nullptr;
    if (natoms < 1 || natoms >= (1 << 20) || nshells < 1 || !coords || !shell_atom || !shell_l || !shell_nprim || !shell_prim_off || !prim_exp ||
        !prim_coef || !aux_exponents)
        return RIS_EINVAL;
    int nprim_tot = 0;
    std::vector<int> shell_ao(nshells);
    int nao = 0;
    for (int s = 0; s < nshells; ++s) {
        if (shell_l[s] < 0 || shell_l[s] > RIS_LMAX || shell_nprim[s] < 1 || shell_nprim[s] > RIS_NPRIM_MAX || shell_atom[s] < 0 ||
            shell_atom[s] >= natoms || shell_prim_off[s] < 0)
            return RIS_EINVAL;
        nprim_tot = std::max(nprim_tot, shell_prim_off[s] + shell_nprim[s]);
        shell_ao[s] = nao;
        nao += ris_ncart(shell_l[s]);
    }
    for (int i = 0; i < 3 * natoms; ++i) if (!std::isfinite(coords[i])) return RIS_EINVAL;
    for (int i = 0; i < nprim_tot; ++i)
        if (!std::isfinite(prim_exp[i]) || !(prim_exp[i] > 0.0) || !std::isfinite(prim_coef[i])) return RIS_EINVAL;
    for (int i = 0; i < natoms; ++i) if (!std::isfinite(aux_exponents[i]) || !(aux_exponents[i] > 0.0)) return RIS_EINVAL;

    int ndev = 0;
    CU(cudaGetDeviceCount(&ndev));
    if (ndev < 1) { g_cuda_err = "no CUDA device (this library has no CPU fallback)"; return RIS_ECUDA; }

    ris_ctx* c = new (std::nothrow) ris_ctx;
    if (!c) return RIS_ENOMEM;
    struct Guard { ris_ctx* c; bool ok = false; ~Guard() { if (!ok) ris_destroy(c); } } guard{c};
    CU(cudaGetDevice(&c->device));
    CU(cudaDeviceGetAttribute(&c->nsm, cudaDevAttrMultiProcessorCount, c->device));
    {   // keep up to 1 GiB of freed packed-pair buffers in the default pool between contexts (the default gives
        // everything back to the driver at the next synchronisation)
        cudaMemPool_t pool;
        CU(cudaDeviceGetDefaultMemPool(&pool, c->device));
        unsigned long long keep = 1ull << 30, cur = 0;
        CU(cudaMemPoolGetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &cur));
        if (cur < keep) CU(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
    }
    c->stream = (cudaStream_t)cuda_stream;
    c->opt.schwarz_tol = 1e-13;
    if (opt) c->opt = *opt;
    c->natoms = natoms; c->nshells = nshells; c->nao = nao; c->naux = natoms;
    c->nao_in = nao;

    int rc;
    if (c->opt.spherical) {
        std::vector<int> sph0((size_t)nao), lc((size_t)nao);
        int ns = 0;
        for (int s = 0; s < nshells; ++s) {
            for (int k = 0; k < ris_ncart(shell_l[s]); ++k) { sph0[shell_ao[s] + k] = ns; lc[shell_ao[s] + k] = 16 * shell_l[s] + k; }
            ns += 2 * shell_l[s] + 1;
        }
        c->nao_in = ns;
        if ((rc = dev_upload(c, &c->d_sph0, sph0.data(), sph0.size()))) return rc;
        if ((rc = dev_upload(c, &c->d_sph_lc, lc.data(), lc.size()))) return rc;
    }
    if ((rc = dev_upload(c, &c->d_coords, coords, (size_t)3 * natoms))) return rc;
    if ((rc = dev_upload(c, &c->d_shell_atom, shell_atom, (size_t)nshells))) return rc;
    if ((rc = dev_upload(c, &c->d_shell_l, shell_l, (size_t)nshells))) return rc;
    if ((rc = dev_upload(c, &c->d_shell_nprim, shell_nprim, (size_t)nshells))) return rc;
    if ((rc = dev_upload(c, &c->d_shell_poff, shell_prim_off, (size_t)nshells))) return rc;
    if ((rc = dev_upload(c, &c->d_shell_ao, shell_ao.data(), (size_t)nshells))) return rc;
    if ((rc = dev_upload(c, &c->d_pexp, prim_exp, (size_t)nprim_tot))) return rc;
    if ((rc = dev_upload(c, &c->d_pcoef, prim_coef, (size_t)nprim_tot))) return rc;

    // aux records (ris_internal.h: RisGradParams::aux) and the potential maximum used by the screening bound
    std::vector<double> aux((size_t)RIS_AUX_FIELDS * natoms);
    double vmax = 0.0;
    for (int P = 0; P < natoms; ++P) {
        aux_record(&aux[(size_t)RIS_AUX_FIELDS * P], coords + 3 * P, aux_exponents[P], 0, 0, P, P);
        vmax = std::max(vmax, std::pow(2.0 * aux_exponents[P] / M_PI, 0.75) * 2.0 * M_PI / aux_exponents[P]);
    }
    if ((rc = dev_upload(c, &c->d_aux, aux.data(), aux.size()))) return rc;
    c->h_coords.assign(coords, coords + 3 * (size_t)natoms);
    c->naux_J = natoms; c->d_jfn = c->d_aux; c->d_jlist[0] = c->d_aux; c->jcnt[0] = natoms;

    // Boys tables, one per top order M = 0..8 (M = 0: the undifferentiated (ss|P) of the fitting step)
    // (geometry-independent: the host tables are built once per process, in long double, and kept)
    {
        static std::vector<double> tabs[9];
        static std::mutex tabs_mu;
        std::lock_guard<std::mutex> lk(tabs_mu);
        for (int M = 0; M <= 8; ++M) {
            if (tabs[M].empty()) ris_build_boys_table(M, RIS_BOYS_NGRID, RIS_BOYS_PER_UNIT, tabs[M]);
            if ((rc = dev_upload(c, &c->d_boys[M], tabs[M].data(), tabs[M].size()))) return rc;
        }
        CU(cudaStreamSynchronize(c->stream));
    }

    // ---- S0 on device: survey -> scan -> scatter -> pack
    // schwarz_tol bounds the ACCUMULATED neglected contribution per unit |D c| or |Gamma| (include/ris.h): the
    // per-primitive-pair threshold is tol / (naux sqrt(number of unique shell pairs)).
    const long long ntot = (long long)nshells * (nshells + 1) / 2;
    const double tol_prim = c->opt.schwarz_tol > 0.0 ? c->opt.schwarz_tol / ((double)natoms * std::sqrt((double)ntot)) : 0.0;
    RisMolDev m{natoms, nshells, c->d_coords, c->d_shell_atom, c->d_shell_l, c->d_shell_nprim, c->d_shell_poff,
                c->d_shell_ao, c->d_pexp, c->d_pcoef, vmax, tol_prim};
    c->npairs_total = ntot;
    for (int i = 0; i <= nshells - 1; ++i)
        for (int j = 0; j <= i; ++j) c->nprim_total += (long long)shell_nprim[i] * shell_nprim[j];
    const int nblk = (int)((ntot + RIS_SCAN_BLOCK - 1) / RIS_SCAN_BLOCK);
    unsigned* d_packed;
    unsigned long long* d_key;
    int *d_hist, *d_base, *d_meta;   // d_meta: totals[16], start[16], kmax[16]
    unsigned long long* d_nprim;
    long long* d_list[2];
    if ((rc = dev_alloc(c, &d_packed, (size_t)ntot, false))) return rc;
    if ((rc = dev_alloc(c, &d_key, (size_t)ntot, false))) return rc;
    if ((rc = dev_alloc(c, &d_hist, (size_t)nblk * RIS_NBIN, false))) return rc;
    if ((rc = dev_alloc(c, &d_base, (size_t)nblk * RIS_NBIN, false))) return rc;
    if ((rc = dev_alloc(c, &d_meta, (size_t)3 * RIS_NBIN, true))) return rc;
    if ((rc = dev_alloc(c, &d_nprim, (size_t)RIS_NBIN, true))) return rc;
    if ((rc = dev_alloc(c, &d_list[0], (size_t)ntot, false))) return rc;
    if ((rc = dev_alloc(c, &d_list[1], (size_t)ntot, false))) return rc;
    {
        ProfScope ps(c, "ris_k_pair_survey");
        ris_k_pair_survey<<<nblk, RIS_SCAN_BLOCK, 0, c->stream>>>(m, ntot, d_packed, d_key, d_meta + 2 * RIS_NBIN, d_nprim);
    }
    // LSD radix sort on (class, atom of mu, atom of nu): 4-bit digits of the atom indices, then the class
    int abits = 1;
    while ((1 << abits) < natoms) ++abits;
    std::vector<int> shifts;
    for (int b = 0; b < abits; b += 4) shifts.push_back(b);
    for (int b = 0; b < abits; b += 4) shifts.push_back(20 + b);
    shifts.push_back(40);
    const long long* lin = nullptr;
    for (size_t pass = 0; pass < shifts.size(); ++pass) {
        ProfScope ps(c, "ris_k_radix_pass");
        long long* lout = d_list[pass & 1];
        ris_k_radix_hist<<<nblk, RIS_SCAN_BLOCK, 0, c->stream>>>(ntot, lin, d_key, shifts[pass], d_hist);
        ris_k_radix_scan<<<1, 32 * RIS_NBIN, 0, c->stream>>>(nblk, d_hist, d_base, d_meta, d_meta + RIS_NBIN);
        ris_k_radix_scatter<<<nblk, RIS_SCAN_BLOCK, 0, c->stream>>>(ntot, lin, d_key, shifts[pass], d_base, d_meta + RIS_NBIN, lout);
        lin = lout;
    }
    const long long* d_sorted = lin;
    CU(cudaGetLastError());
    int meta[3 * RIS_NBIN];
    unsigned long long nprim_c[RIS_NBIN];
    CU(cudaMemcpyAsync(meta, d_meta, sizeof meta, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaMemcpyAsync(nprim_c, d_nprim, sizeof nprim_c, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));

    long long off = 0;
    for (int la = 0; la <= RIS_LMAX; ++la)
        for (int lb = 0; lb <= la; ++lb) {
            const int k = ris_class_id(la, lb);
            RisClassPack& pk = c->cls[k];
            pk.la = la; pk.lb = lb;
            pk.npairs = meta[k];
            pk.kmax = meta[2 * RIS_NBIN + k];
            pk.nprim = (long long)nprim_c[k];
            pk.task_prims = ris_task_prims(la, lb);
            pk.ntasks = (int)((pk.nprim + pk.task_prims - 1) / pk.task_prims);
            pk.elem_off = off;
            off += (long long)ris_ncart(la) * ris_ncart(lb) * pk.npairs;
            c->nprim_surv += pk.nprim;
            if (pk.npairs == 0) continue;
            const size_t n = (size_t)pk.npairs;
            if ((rc = dev_alloc(c, &pk.pairs, n, false))) return rc;
            if ((rc = dev_alloc(c, &pk.ao, 2 * n, false))) return rc;
            if ((rc = dev_alloc(c, &pk.symf, n, false))) return rc;
            if ((rc = dev_alloc(c, &pk.prim_off, n + 1, false))) return rc;
            if ((rc = dev_alloc(c, &pk.prim, (size_t)pk.nprim * RIS_PRIM_FIELDS, false))) return rc;
            if ((rc = dev_alloc(c, &pk.task_begin, (size_t)pk.ntasks + 1, false))) return rc;
            ProfScope ps(c, "ris_k_pair_pack");
            ris_k_scan_nk<<<1, 1024, 0, c->stream>>>(pk.npairs, d_sorted + meta[RIS_NBIN + k], d_packed, pk.prim_off);
            ris_k_task_bounds<<<(pk.ntasks + 1 + 127) / 128, 128, 0, c->stream>>>(pk.npairs, pk.ntasks, pk.task_prims, pk.prim_off, pk.task_begin);
            ris_k_pair_pack<<<(pk.npairs + 127) / 128, 128, 0, c->stream>>>(m, pk, d_sorted + meta[RIS_NBIN + k]);
        }
    c->nelem_real = off;
    CU(cudaGetLastError());
    {   // "small": no class fills the GPU with its one resident wave (the criterion of launch_classes for the default set)
        long long most = 0;
        const int ny = (natoms + 31) / 32;
        for (int k = 0; k < RIS_NCLASS; ++k)
            if (c->cls[k].npairs > 0) most = std::max(most, (long long)((c->cls[k].ntasks + RIS_GRAD_WARPS - 1) / RIS_GRAD_WARPS) * ny);
        // ... AND little work altogether (under 1e7 primitive triplets: a call of well under a millisecond, where launch and
        // dependency latency is what is being paid).  Config 5 (40 atoms with f shells, 5 ms per call) has few tasks per class
        // but nothing to gain from a graph; its end-to-end call was measured slower and erratic with one (6.0 -> 6.7-11 ms).
        c->small = most <= (long long)2 * c->nsm && c->nprim_surv * (long long)natoms < 10000000ll &&
                   !std::getenv("RIS_NO_GRAPH");                                  // (the variable: A/B measurements)
    }
    // spatial AO order + block list for the pair-restricted Gamma^P GEMM-2
    {
        double lo[3] = {coords[0], coords[1], coords[2]};
        for (int a = 0; a < natoms; ++a)
            for (int d = 0; d < 3; ++d) lo[d] = std::min(lo[d], coords[3 * a + d]);
        std::vector<std::pair<unsigned long long, int>> key(natoms);
        for (int a = 0; a < natoms; ++a) key[a] = {morton3(coords + 3 * a, lo), a};
        std::sort(key.begin(), key.end());
        std::vector<int> arank(natoms);
        for (int i = 0; i < natoms; ++i) arank[key[i].second] = i;
        std::vector<int> sh(nshells);
        for (int i = 0; i < nshells; ++i) sh[i] = i;
        std::stable_sort(sh.begin(), sh.end(), [&](int x, int y) { return arank[shell_atom[x]] < arank[shell_atom[y]]; });
        std::vector<int> ao_pos(nao), ao_order(nao);
        int pos = 0;
        for (int i = 0; i < nshells; ++i)
            for (int k = 0; k < ris_ncart(shell_l[sh[i]]); ++k) { ao_pos[shell_ao[sh[i]] + k] = pos; ao_order[pos] = shell_ao[sh[i]] + k; ++pos; }
        if ((rc = dev_upload(c, &c->d_ao_pos, ao_pos.data(), ao_pos.size()))) return rc;
        if ((rc = dev_upload(c, &c->d_ao_order, ao_order.data(), ao_order.size()))) return rc;
        c->nblk = (nao + RIS_GTILE2 - 1) / RIS_GTILE2;
        // GEMM-2 partner lists and the fit_K bands, built on the device (two small D2H reads: tile count, band ranges)
        constexpr int BM = RIS_G2_BM;
        int *d_cnt, *d_tbase, *d_fill, *d_jlo, *d_jhi;
        if ((rc = dev_alloc(c, &d_cnt, (size_t)nao, true))) return rc;
        if ((rc = dev_alloc(c, &d_fill, (size_t)nao, true))) return rc;
        if ((rc = dev_alloc(c, &d_tbase, (size_t)nao + 1, true))) return rc;
        if ((rc = dev_alloc(c, &d_jlo, (size_t)c->nblk, false))) return rc;
        if ((rc = dev_alloc(c, &d_jhi, (size_t)c->nblk, false))) return rc;
        CU(cudaMemsetAsync(d_jlo, 0x7f, sizeof(int) * (size_t)c->nblk, c->stream));
        CU(cudaMemsetAsync(d_jhi, 0xff, sizeof(int) * (size_t)c->nblk, c->stream));
        for (int k = 0; k < RIS_NCLASS; ++k) {
            const RisClassPack& pk = c->cls[k];
            if (pk.npairs == 0) continue;
            const long long nelc = (long long)ris_ncart(pk.la) * ris_ncart(pk.lb) * pk.npairs;
            ris_k_g2_count<<<(unsigned)((nelc + 255) / 256), 256, 0, c->stream>>>(pk, c->d_ao_pos, d_cnt, d_jlo, d_jhi);
        }
        ris_k_g2_scan<<<1, 1024, 0, c->stream>>>(nao, BM, d_cnt, d_tbase);
        CU(cudaGetLastError());
        std::vector<int> jlo(c->nblk), jhi(c->nblk);
        CU(cudaMemcpyAsync(&c->ntiles, d_tbase + nao, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaMemcpyAsync(jlo.data(), d_jlo, sizeof(int) * (size_t)c->nblk, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaMemcpyAsync(jhi.data(), d_jhi, sizeof(int) * (size_t)c->nblk, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        c->g2_entries = 2 * c->nelem_real;
        const size_t nrow = (size_t)std::max(c->ntiles, 1) * BM;
        if ((rc = dev_alloc(c, &c->d_g2tiles, (size_t)std::max(c->ntiles, 1), false))) return rc;
        if ((rc = dev_alloc(c, &c->d_g2rows, nrow, false))) return rc;
        if ((rc = dev_alloc(c, &c->d_g2code, nrow, false))) return rc;
        CU(cudaMemsetAsync(c->d_g2rows, 0xff, sizeof(int) * nrow, c->stream));
        CU(cudaMemsetAsync(c->d_g2code, 0xff, sizeof(int) * nrow, c->stream));
        for (int k = 0; k < RIS_NCLASS; ++k) {
            const RisClassPack& pk = c->cls[k];
            if (pk.npairs == 0) continue;
            const long long nelc = (long long)ris_ncart(pk.la) * ris_ncart(pk.lb) * pk.npairs;
            ris_k_g2_fill<<<(unsigned)((nelc + 255) / 256), 256, 0, c->stream>>>(pk, c->d_ao_pos, BM, d_tbase, d_fill, c->d_g2rows, c->d_g2code);
        }
        ris_k_g2_tiles<<<(nao + 127) / 128, 128, 0, c->stream>>>(nao, BM, d_tbase, c->d_g2tiles);
        CU(cudaGetLastError());
        {   // row-block bands for the fitting step's sparse transform (ris_fit_K)
            c->rb_jlo.resize(c->nblk); c->rb_kw.resize(c->nblk); c->rb_off.resize(c->nblk);
            long long off2 = 0;
            for (int I = 0; I < c->nblk; ++I) {
                if (jhi[I] < 0 || jlo[I] > jhi[I]) jlo[I] = jhi[I] = I;
                c->rb_jlo[I] = jlo[I]; c->rb_kw[I] = (jhi[I] - jlo[I] + 1) * RIS_GTILE2; c->rb_off[I] = off2;
                off2 += (long long)RIS_GTILE2 * c->rb_kw[I];
            }
            c->slab_stride = off2;
            if ((rc = dev_upload(c, &c->d_rb_jlo, c->rb_jlo.data(), c->rb_jlo.size()))) return rc;
            if ((rc = dev_upload(c, &c->d_rb_kw, c->rb_kw.data(), c->rb_kw.size()))) return rc;
            if ((rc = dev_upload(c, &c->d_rb_off, c->rb_off.data(), c->rb_off.size()))) return rc;
        }
        CU(cudaStreamSynchronize(c->stream));      // host vectors go out of scope
    }
    CU(cudaStreamSynchronize(c->stream));
    guard.ok = true;
    *out = c;
    return RIS_OK;
}

extern "C" int ris_destroy(ris_ctx* c)
{
    if (!c) return RIS_EINVAL;
    cudaStreamSynchronize(c->stream);
    graphs_invalidate(c);
    ris_resp_free(c);
    for (void* p : c->owned) cudaFreeAsync(p, c->stream);
    cudaStreamSynchronize(c->stream);
    for (int i = 0; i < WS_N; ++i) if (c->ws[i]) cudaFree(c->ws[i]);
    for (cudaEvent_t e : c->copy_ev) cudaEventDestroy(e);
    if (c->copy_gate) cudaEventDestroy(c->copy_gate);
    if (c->copy_extra) cudaEventDestroy(c->copy_extra);
    if (c->fork_ev) cudaEventDestroy(c->fork_ev);
    for (int k = 0; k < RIS_NCLASS; ++k) {
        if (c->join_ev[k]) cudaEventDestroy(c->join_ev[k]);
        if (c->side[k]) cudaStreamDestroy(c->side[k]);
        if (c->join2_ev[k]) cudaEventDestroy(c->join2_ev[k]);
        if (c->side2[k]) cudaStreamDestroy(c->side2[k]);
    }
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    ris_profile_reset(c);
    delete c;
    return RIS_OK;
}

extern "C" int ris_nao(const ris_ctx* c) { return c ? c->nao_in : RIS_EINVAL; }
extern "C" int ris_naux(const ris_ctx* c) { return c ? c->naux : RIS_EINVAL; }
extern "C" int ris_natoms(const ris_ctx* c) { return c ? c->natoms : RIS_EINVAL; }
extern "C" long long ris_npairs(const ris_ctx* c, int la, int lb)
{
    if (!c || la < lb || la > RIS_LMAX || lb < 0) return RIS_EINVAL;
    return c->cls[ris_class_id(la, lb)].npairs;
}
extern "C" long long ris_nprimpairs(const ris_ctx* c, int la, int lb)
{
    if (!c || la < lb || la > RIS_LMAX || lb < 0) return RIS_EINVAL;
    return c->cls[ris_class_id(la, lb)].nprim;
}
extern "C" long long ris_npairs_total(const ris_ctx* c) { return c ? c->npairs_total : RIS_EINVAL; }
extern "C" long long ris_ntriplets(const ris_ctx* c) { return c ? c->nprim_surv * c->naux : RIS_EINVAL; }
extern "C" long long ris_ntriplets_unscreened(const ris_ctx* c) { return c ? c->nprim_total * c->naux : RIS_EINVAL; }
extern "C" long long ris_npair_elements(const ris_ctx* c) { return c ? c->nelem_real : RIS_EINVAL; }
extern "C" int ris_p_batch(const ris_ctx* c) { return c ? c->last_pbatch : RIS_EINVAL; }

// Spherical mode (ris_sph.cuh): the caller's coefficient matrix [nao_in][ncol] expanded to Cartesian rows [nao][ncol] in a
// ctx-owned buffer; Cartesian mode hands the pointer through.
static int sph_coef(ris_ctx* c, int slot, const double* C, int ncol, const double** out)
{
    *out = C;
    if (!c->opt.spherical) return RIS_OK;
    double* w;
    int rc = ws_get(c, slot, sizeof(double) * (size_t)c->nao * ncol, (void**)&w);
    if (rc) return rc;
    const long long n = (long long)c->nao * ncol;
    {
        ProfScope ps(c, "ris_k_sph_coef", 2.0 * n, 16.0 * n);
        ris_k_sph_coef<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->nao, ncol, c->d_sph0, c->d_sph_lc, C, w);
    }
    CU(cudaGetLastError());
    *out = w;
    return RIS_OK;
}

// --------------------------------------------------------------------------------------- tile packing
// J tiles: out[slab][elem_off + ip*nel + e] = symf[ip] * (G[slab][mu0+ca][nu0+cb] + G[slab][nu0+cb][mu0+ca]),  e = ca*ncb + cb.
// Folds D + D^T onto the unique shell pairs.
// One launch for all classes: blockIdx.y selects the class (sph0 != nullptr: spherical mode, ris_sph.cuh).
struct RisPackAll { RisClassPack pk[RIS_NCLASS]; int ncls; };
__global__ void ris_k_pack_tiles(RisPackAll pa, int nao, const int* __restrict__ sph0, const double* __restrict__ G, long long gstride,
                                 double* __restrict__ out, long long ostride)
{
    const RisClassPack& pk = pa.pk[blockIdx.y];
    const int nca = ris_ncart(pk.la), ncb = ris_ncart(pk.lb), nel = nca * ncb;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)pk.npairs * nel) return;
    const int ip = (int)(idx / nel), e = (int)(idx - (long long)ip * nel), ca = e / ncb, cb = e - ca * ncb;
    const double* g = G + (size_t)blockIdx.z * gstride;
    double v;
    if (sph0 == nullptr) {
        const size_t r = (size_t)pk.ao[ip] + ca, q = (size_t)pk.ao[(size_t)pk.npairs + ip] + cb;
        v = g[r * nao + q] + g[q * nao + r];
    } else {
        v = ris_sph_pair_element(pk.la, pk.lb, ca, cb, (size_t)sph0[pk.ao[ip]], (size_t)sph0[pk.ao[(size_t)pk.npairs + ip]], nao, g);
    }
    out[(size_t)blockIdx.z * ostride + pk.elem_off + idx] = (double)pk.symf[ip] * v;
}

static int pack_tiles(ris_ctx* c, const double* G, long long gstride, int nslab, double* out, long long ostride)
{
    RisPackAll pa{};
    long long most = 0;
    double nel = 0.0;
    for (int k = 0; k < RIS_NCLASS; ++k) {
        const RisClassPack& pk = c->cls[k];
        if (pk.npairs == 0) continue;
        pa.pk[pa.ncls++] = pk;
        const long long n = (long long)ris_ncart(pk.la) * ris_ncart(pk.lb) * pk.npairs;
        most = std::max(most, n);
        nel += (double)n;
    }
    if (pa.ncls == 0) return RIS_OK;
    ProfScope ps(c, "ris_k_pack_tiles", 2.0 * nel * nslab, 24.0 * nel * nslab);
    dim3 grid((unsigned)((most + 255) / 256), pa.ncls, nslab);
    ris_k_pack_tiles<<<grid, 256, 0, c->stream>>>(pa, c->opt.spherical ? c->nao_in : c->nao, c->opt.spherical ? c->d_sph0 : nullptr, G,
                                                  gstride, out, ostride);
    CU(cudaGetLastError());
    return RIS_OK;
}

// One launch per class, heaviest class first.  tile / sstride / estride / lstride: see RisGradParams.
// aux / aux_type / naux_row: the list of auxiliary functions of this pass (records, type 0 = s, 1..3 = p_x..p_z) and the row
// length of cscale; [p0, p1) = range of list positions.
static int launch_classes(ris_ctx* c, const double* tile, long long sstride, long long estride, int lstride,
                          const double* cscale, int nb, int p0, int p1, double* grad, unsigned long long* det,
                          const double* aux = nullptr, int aux_type = 0, int naux_row = 0)
{
    if (!aux) { aux = c->d_aux; naux_row = c->naux; }
    const int eb = aux_type ? 2 : 1;       // Boys order above la + lb: the derivative, and the step on a p aux centre
    const int ny = (p1 - p0 + 31) / 32;
    int* ctr;
    // two ticket arrays per class: the heavy classes run their host-centre phases as two launches
    { int rc = ws_get(c, WS_CTR, sizeof(int) * (size_t)2 * RIS_NCLASS * ny, (void**)&ctr); if (rc) return rc; }
    CU(cudaMemsetAsync(ctr, 0, sizeof(int) * (size_t)2 * RIS_NCLASS * ny, c->stream));
    // Small molecules: no class has enough warp tasks to fill the GPU with its one resident wave, so the class kernels
    // run side by side on their own streams (fork from / join into the context's stream); large ones run back to back.
    const int nsm = c->nsm;
    long long most = 0;
    int nclass = 0;
    for (int k = 0; k < RIS_NCLASS; ++k)
        if (c->cls[k].npairs > 0) { most = std::max(most, (long long)((c->cls[k].ntasks + RIS_GRAD_WARPS - 1) / RIS_GRAD_WARPS) * ny); ++nclass; }
    const bool side = nclass > 1 && most <= (long long)2 * nsm;
    if (side) {
        if (!c->fork_ev) CU(cudaEventCreateWithFlags(&c->fork_ev, cudaEventDisableTiming));
        for (int k = 0; k < RIS_NCLASS; ++k)
            if (!c->side[k]) {
                CU(cudaStreamCreateWithFlags(&c->side[k], cudaStreamNonBlocking));
                CU(cudaEventCreateWithFlags(&c->join_ev[k], cudaEventDisableTiming));
                CU(cudaStreamCreateWithFlags(&c->side2[k], cudaStreamNonBlocking));
                CU(cudaEventCreateWithFlags(&c->join2_ev[k], cudaEventDisableTiming));
            }
        CU(cudaEventRecord(c->fork_ev, c->stream));
    }
    for (int oi = 0; oi < RIS_NCLASS; ++oi) {
        const int k = kClassOrder[oi];
        const RisClassPack& pk = c->cls[k];
        if (pk.npairs == 0) continue;
        const cudaStream_t st = side ? c->side[k] : c->stream;
        const bool two = side && ris_grad_split(pk.la, pk.lb);     // the second host phase of a split class on its own stream
        if (side) CU(cudaStreamWaitEvent(st, c->fork_ev, 0));
        if (two) CU(cudaStreamWaitEvent(c->side2[k], c->fork_ev, 0));
        RisGradParams p{};
        p.phase2_stream = two ? c->side2[k] : nullptr;
        p.task_ctr = ctr + (size_t)2 * k * ny;
        p.pk = pk; p.naux = naux_row; p.natoms = c->natoms; p.nsm = c->nsm; p.aux = aux; p.aux_type = aux_type;
        p.boys = c->d_boys[pk.la + pk.lb + eb];
        p.tile = tile; p.sstride = sstride; p.estride = estride; p.lstride = lstride; p.cscale = cscale; p.nb = nb;
        p.p0 = p0; p.p1 = p1;
        p.grad = grad; p.det = det; p.det_flag = det ? (int*)c->ws[WS_DET] : nullptr;
        const double np_ = (double)(p1 - p0), nel = (double)ris_ncart(pk.la) * ris_ncart(pk.lb);
        {
            ProfScope ps(c, kGradNames[k], np_ * ((double)pk.nprim * kModelFlopsByE[pk.la + pk.lb + eb] + 12.0 * nel * pk.npairs * nb),
                         8.0 * (lstride ? np_ : 1.0) * nel * pk.npairs * nb + 8.0 * (double)pk.nprim * RIS_PRIM_FIELDS, st, false);
            CU(ris_grad_launchers[k](p, st));
        }
        if (side) {
            CU(cudaEventRecord(c->join_ev[k], st));
            CU(cudaStreamWaitEvent(c->stream, c->join_ev[k], 0));
        }
        if (two) {
            CU(cudaEventRecord(c->join2_ev[k], c->side2[k]));
            CU(cudaStreamWaitEvent(c->stream, c->join2_ev[k], 0));
        }
    }
    CU(cudaGetLastError());
    return RIS_OK;
}

// states per class-kernel launch: as even as possible, at most `cap` (<= RIS_NB_MAX)
static int next_nb(int remaining, int cap)
{
    const int launches = (remaining + cap - 1) / cap;
    return (remaining + launches - 1) / launches;
}
// the cap: every class present must fit its block into shared memory (long contractions: kmax up to 576 records per task)
static int nb_cap(const ris_ctx* c, bool ktype)
{
    int cap = RIS_NB_MAX;
    for (int k = 0; k < RIS_NCLASS; ++k)
        if (c->cls[k].npairs > 0) cap = std::min(cap, ris_grad_nb_cap(c->cls[k].la, c->cls[k].lb, c->cls[k].kmax, ktype));
    return cap;
}

// --------------------------------------------------------------------------------------- deterministic reduction
// grad[i] = hi[i] 2^-28 + lo[i] 2^-60 (ris_internal.h: ris_grad_add); NaN everywhere when a contribution left the range.
__global__ void ris_k_det_finish(long long n, const unsigned long long* __restrict__ acc, const int* __restrict__ flag,
                                 double* __restrict__ grad)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double v = (double)(long long)acc[2 * i] * (1.0 / 268435456.0) + (double)(long long)acc[2 * i + 1] * (1.0 / 1152921504606846976.0);
    grad[i] = *flag ? nan("") : v;
}

// Layout of WS_DET: int flag (16 bytes reserved), then [nbatch][natoms][3][2] accumulators.
static int det_begin(ris_ctx* c, int nbatch, unsigned long long** acc)
{
    *acc = nullptr;
    if (!c->opt.deterministic) return RIS_OK;
    void* w;
    const size_t bytes = 16 + sizeof(unsigned long long) * 2 * (size_t)nbatch * c->natoms * 3;
    int rc = ws_get(c, WS_DET, bytes, &w);
    if (rc) return rc;
    CU(cudaMemsetAsync(w, 0, bytes, c->stream));
    *acc = (unsigned long long*)((char*)w + 16);
    return RIS_OK;
}

static int det_end(ris_ctx* c, int nbatch, const unsigned long long* acc, double* grad)
{
    if (!acc) return RIS_OK;
    const long long n = (long long)nbatch * c->natoms * 3;
    ProfScope ps(c, "ris_k_det_finish", 2.0 * n, 24.0 * n);
    ris_k_det_finish<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(n, acc, (const int*)c->ws[WS_DET], grad);
    CU(cudaGetLastError());
    return RIS_OK;
}

// --------------------------------------------------------------------------------------- J
// Small molecules are bound by launch and cross-stream dependency latency (config 2: ~25 launches on up to 17 streams for
// 0.15 ms of kernels).  A device-pointer call whose signature (arguments and sizes) repeats is therefore captured into a CUDA
// graph on its second occurrence -- the ordinary launch sequence, recorded instead of run -- and replayed afterwards; a call
// with a new signature runs directly and replaces the remembered one.  Not used while profiling, inside a capture of the
// caller's own, or for molecules that fill the GPU (nothing to gain there).
template <class F>
static int run_graphed(ris_ctx* c, int slot, const std::vector<unsigned long long>& key, F&& body)
{
    if (!c->small || c->opt.profile) return body();
    ris_ctx::GraphSlot& g = c->gslot[slot];
    if (g.exec && g.key == key) { CU(cudaGraphLaunch(g.exec, c->stream)); return RIS_OK; }
    if (g.key != key) {                               // first sight of this signature: run it, remember it
        if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
        const int rc = body();
        if (rc == RIS_OK) g.key = key; else g.key.clear();
        return rc;
    }
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    CU(cudaSetDevice(c->device));
    if (cudaStreamIsCapturing(c->stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) { cudaGetLastError(); return body(); }
    if (!c->cap_stream) CU(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
    const cudaStream_t user = c->stream;
    c->stream = c->cap_stream;                        // the launch sequence below is recorded on our stream ...
    cudaError_t e = cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed);
    if (e != cudaSuccess) { cudaGetLastError(); c->stream = user; g.key.clear(); return body(); }
    const int rc = body();
    cudaGraph_t graph = nullptr;
    e = cudaStreamEndCapture(c->stream, &graph);
    c->stream = user;                                 // ... and replayed in the caller's
    if (rc != RIS_OK || e != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        g.key.clear();
        return rc != RIS_OK ? rc : body();            // capture refused: run directly
    }
    const cudaError_t ei = cudaGraphInstantiate(&g.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ei != cudaSuccess) { cudaGetLastError(); g.exec = nullptr; g.key.clear(); return body(); }
    CU(cudaGraphLaunch(g.exec, c->stream));
    return RIS_OK;
}
static inline unsigned long long key_of(const void* p) { return (unsigned long long)(uintptr_t)p; }

static int grad_J_impl(ris_ctx* c, int nbatch, const double* D, const double* c_aux, double* grad, int f_lo, int f_hi);
static int grad_J_graphed(ris_ctx* c, int nbatch, const double* D, const double* c_aux, double* grad, int f_lo, int f_hi)
{
    const std::vector<unsigned long long> key = {1ull, (unsigned long long)nbatch, key_of(D), key_of(c_aux), key_of(grad),
                                                 (unsigned long long)f_lo, (unsigned long long)f_hi};
    return run_graphed(c, 0, key, [&]() { return grad_J_impl(c, nbatch, D, c_aux, grad, f_lo, f_hi); });
}
extern "C" int ris_grad_J(ris_ctx* c, int nbatch, const double* D, const double* c_aux, double* grad)
{
    return c ? grad_J_graphed(c, nbatch, D, c_aux, grad, 0, c->naux_J) : RIS_EINVAL;
}
extern "C" int ris_grad_J_range(ris_ctx* c, int nbatch, const double* D, const double* c_aux, int f_lo, int f_hi, double* grad)
{
    return c ? grad_J_graphed(c, nbatch, D, c_aux, grad, f_lo, f_hi) : RIS_EINVAL;
}

// [f_lo, f_hi): the J-fit FUNCTIONS this call sums over (c_aux keeps its full row length)
static int grad_J_impl(ris_ctx* c, int nbatch, const double* D, const double* c_aux, double* grad, int f_lo, int f_hi)
{
    if (!c || nbatch < 1 || !D || !c_aux || !grad || f_lo < 0 || f_hi > c->naux_J || f_lo > f_hi) return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    CU(cudaMemsetAsync(grad, 0, sizeof(double) * (size_t)nbatch * c->natoms * 3, c->stream));
    const long long nao2 = (long long)c->nao_in * c->nao_in;
    unsigned long long* det;
    { int rc = det_begin(c, nbatch, &det); if (rc) return rc; }
    const int cap = nb_cap(c, false);
    if (cap < 1) return RIS_ENOMEM;
    for (int s0 = 0, nb; s0 < nbatch; s0 += nb) {
        nb = next_nb(nbatch - s0, cap);
        double* tile;
        int rc = ws_get(c, WS_TILE, sizeof(double) * (size_t)nb * c->nelem_real, (void**)&tile);
        if (rc) return rc;
        if ((rc = pack_tiles(c, D + (size_t)s0 * nao2, nao2, nb, tile, c->nelem_real))) return rc;
        for (int t = 0; t < 4; ++t) {       // one pass per type of auxiliary function: s, p_x, p_y, p_z
            // list positions whose function index lies in [f_lo, f_hi): the lists are in ascending function order
            int q0 = 0, q1 = c->jcnt[t];
            if (c->jfit) {
                const std::vector<int>& fn = c->h_jlist_fn[t];
                q0 = (int)(std::lower_bound(fn.begin(), fn.end(), f_lo) - fn.begin());
                q1 = (int)(std::lower_bound(fn.begin(), fn.end(), f_hi) - fn.begin());
            } else if (t == 0) {            // default set: the s list IS the function order; there are no p lists
                q0 = f_lo; q1 = f_hi;
            } else {
                q0 = q1 = 0;
            }
            if (q1 > q0 &&
                (rc = launch_classes(c, tile, c->nelem_real, 1, 0, c_aux + (size_t)s0 * c->naux_J, nb, q0, q1,
                                     grad + (size_t)s0 * c->natoms * 3, det ? det + (size_t)2 * s0 * c->natoms * 3 : nullptr,
                                     c->d_jlist[t], t, c->naux_J)))
                return rc;
        }
    }
    return det_end(c, nbatch, det, grad);
}

// --------------------------------------------------------------------------------------- fitting step, J type (NEXT-1)
// M[P][Q] = N_P N_Q (P|Q) = fP fQ 2 pi^{5/2} / sqrt(alpha+beta) F_0(rho R^2), fP = N_P / alpha   (Eq. 22)
__global__ void ris_k_metric(int n, const double* __restrict__ aux, const double* __restrict__ boys0, double* __restrict__ M)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n * n) return;
    const int P = (int)(t / n), Q = (int)(t - (long long)P * n);
    const double X0 = aux[RIS_AUX_FIELDS * P] - aux[RIS_AUX_FIELDS * Q], X1 = aux[RIS_AUX_FIELDS * P + 1] - aux[RIS_AUX_FIELDS * Q + 1], X2 = aux[RIS_AUX_FIELDS * P + 2] - aux[RIS_AUX_FIELDS * Q + 2];
    const double al = aux[RIS_AUX_FIELDS * P + 3], be = aux[RIS_AUX_FIELDS * Q + 3];
    const double sI = ris_rsqrt(al + be);
    double F[1];
    ris_boys<0>(al * be * sI * sI * (X0 * X0 + X1 * X1 + X2 * X2), boys0, F);
    M[t] = aux[RIS_AUX_FIELDS * P + 4] * aux[RIS_AUX_FIELDS * Q + 4] * (2.0 * 17.493418327624862846) * sI * F[0];
}

// In-place Cholesky factor M = L L^T (lower triangle) by ONE block, right-looking, column by column: naux = natoms is a
// few hundred to a few thousand, the factorisation runs once per geometry.  flag = 1 when a pivot is not positive.
__global__ void __launch_bounds__(1024) ris_k_cholesky(int n, double* __restrict__ M, int* flag)
{
    __shared__ double piv, dmax;
    if (threadIdx.x == 0) {
        double m = 0.0;
        for (int j = 0; j < n; ++j) m = fmax(m, M[(size_t)j * n + j]);
        dmax = m;
    }
    __syncthreads();
    for (int j = 0; j < n; ++j) {
        if (threadIdx.x == 0) {
            const double d = M[(size_t)j * n + j];
            if (!(d > 1e-12 * dmax)) *flag = 1;        // numerically singular: (nearly) coincident aux functions
            piv = sqrt(d);
            M[(size_t)j * n + j] = piv;
        }
        __syncthreads();
        const double inv = 1.0 / piv;
        for (int i = j + 1 + threadIdx.x; i < n; i += blockDim.x) M[(size_t)i * n + j] *= inv;
        __syncthreads();
        // trailing update of the lower triangle: M[i][k] -= L[i][j] L[k][j], j < k <= i; thread -> row i, k runs along the row
        const int m = n - j - 1;
        for (long long t = threadIdx.x; t < (long long)m * m; t += blockDim.x) {
            const int i = j + 1 + (int)(t / m), k = j + 1 + (int)(t % m);
            if (k <= i) M[(size_t)i * n + k] = fma(-M[(size_t)i * n + j], M[(size_t)k * n + j], M[(size_t)i * n + k]);
        }
        __syncthreads();
    }
}

// c[s] = (L L^T)^-1 v[s]: one block per state, column-oriented forward and backward substitution in shared memory.
__global__ void __launch_bounds__(256) ris_k_chol_solve(int n, const double* __restrict__ L, const double* __restrict__ v,
                                                        double* __restrict__ cout)
{
    extern __shared__ double y[];
    const int s = blockIdx.x;
    for (int i = threadIdx.x; i < n; i += blockDim.x) y[i] = v[(size_t)s * n + i];
    __syncthreads();
    for (int j = 0; j < n; ++j) {
        if (threadIdx.x == 0) y[j] /= L[(size_t)j * n + j];
        __syncthreads();
        const double yj = y[j];
        for (int i = j + 1 + threadIdx.x; i < n; i += blockDim.x) y[i] = fma(-L[(size_t)i * n + j], yj, y[i]);
        __syncthreads();
    }
    for (int j = n - 1; j >= 0; --j) {
        if (threadIdx.x == 0) y[j] /= L[(size_t)j * n + j];
        __syncthreads();
        const double yj = y[j];
        for (int i = threadIdx.x; i < j; i += blockDim.x) y[i] = fma(-L[(size_t)j * n + i], yj, y[i]);
        __syncthreads();
    }
    for (int i = threadIdx.x; i < n; i += blockDim.x) cout[(size_t)s * n + i] = y[i];
}

// ---- two-centre integrals over the s and p functions of an explicit J-fit set (NEXT-2; Eq. 22) ----
// p_i(r; C, alpha) = (r - C)_i exp(-alpha |r-C|^2) = (1/2 alpha) d/dC_i of the s primitive, so with R = C_f - C_g and
// V(R) = F_0(rho R^2):  (f|g) = N_f N_g 2 pi^{5/2}/(alpha beta sqrt(alpha+beta)) (1/2 alpha)^{l_f} (-1/2 beta)^{l_g} d_i^{l_f} d_j^{l_g} V,
// and d/dC_f adds one more d_k.  Cartesian derivatives of V, with G_n = (-2 rho)^n F_n(rho R^2):
//   d_a V = X_a G_1;  d_a d_b V = X_a X_b G_2 + delta_ab G_1;
//   d_a d_b d_c V = X_a X_b X_c G_3 + (delta_ab X_c + delta_ac X_b + delta_bc X_a) G_2.
RIS_DEV double ris_dV(int n, const int* d, const double* X, const double* G)
{
    if (n == 0) return G[0];
    if (n == 1) return X[d[0]] * G[1];
    if (n == 2) return fma(X[d[0]] * X[d[1]], G[2], d[0] == d[1] ? G[1] : 0.0);
    const double t = (d[0] == d[1] ? X[d[2]] : 0.0) + (d[0] == d[2] ? X[d[1]] : 0.0) + (d[1] == d[2] ? X[d[0]] : 0.0);
    return fma(X[d[0]] * X[d[1]] * X[d[2]], G[3], t * G[2]);
}

struct RisAuxFn { double C[3], al, fac; int atom, fn, l, comp; };
RIS_DEV RisAuxFn ris_aux_fn(const double* __restrict__ rec, int f)
{
    const double* r = rec + (size_t)RIS_AUX_FIELDS * f;
    RisAuxFn a;
    a.C[0] = r[0]; a.C[1] = r[1]; a.C[2] = r[2]; a.al = r[3]; a.fac = r[4];
    const int2 i0 = *reinterpret_cast<const int2*>(r + 5), i1 = *reinterpret_cast<const int2*>(r + 6);
    a.atom = i0.x; a.fn = i0.y; a.l = i1.x; a.comp = i1.y;
    return a;
}

// common factor and direction list of the pair (f, g); returns the number of directions
RIS_DEV int ris_pair_fg(const RisAuxFn& f, const RisAuxFn& g, double* X, int* d, double& pref, double& rho)
{
    X[0] = f.C[0] - g.C[0]; X[1] = f.C[1] - g.C[1]; X[2] = f.C[2] - g.C[2];
    const double sI = ris_rsqrt(f.al + g.al);
    rho = f.al * g.al * sI * sI;
    pref = f.fac * g.fac * (2.0 * 17.493418327624862846) * sI;
    int n = 0;
    if (f.l) { d[n++] = f.comp; pref *= 0.5 / f.al; }
    if (g.l) { d[n++] = g.comp; pref *= -0.5 / g.al; }
    return n;
}

__global__ void ris_k_metric_fn(int n, const double* __restrict__ rec, const double* __restrict__ boys2, double* __restrict__ M)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n * n) return;
    const RisAuxFn f = ris_aux_fn(rec, (int)(t / n)), g = ris_aux_fn(rec, (int)(t % n));
    double X[3], pref, rho, F[3];
    int d[3];
    const int nd = ris_pair_fg(f, g, X, d, pref, rho);
    ris_boys<2>(rho * (X[0] * X[0] + X[1] * X[1] + X[2] * X[2]), boys2, F);
    const double G[3] = {F[0], -2.0 * rho * F[1], 4.0 * rho * rho * F[2]};
    M[t] = pref * ris_dV(nd, d, X, G);
}

// g[s][A] = sum_{f on A} sum_{g not on A} (c_f d_g + c_g d_f) d(f|g)/dC_f: one block per (atom, state), the atom's functions
// in list order, threads over g, fixed-order block reduction (deterministic).  Pairs on one atom move together: no term.
__global__ void __launch_bounds__(128) ris_k_grad_pq_fn(int n, const double* __restrict__ rec, const int* __restrict__ afo,
                                                        const int* __restrict__ afn, const double* __restrict__ boys3,
                                                        const double* __restrict__ cv, const double* __restrict__ dv,
                                                        double* __restrict__ grad)
{
    const int A = blockIdx.x, s = blockIdx.y;
    double acc[3] = {0.0, 0.0, 0.0};
    for (int k = afo[A]; k < afo[A + 1]; ++k) {
        const RisAuxFn f = ris_aux_fn(rec, afn[k]);
        const double cf = cv[(size_t)s * n + f.fn], df = dv[(size_t)s * n + f.fn];
        for (int q = threadIdx.x; q < n; q += blockDim.x) {
            const RisAuxFn g = ris_aux_fn(rec, q);
            if (g.atom == A) continue;
            double X[3], pref, rho, F[4];
            int d[3];
            const int nd = ris_pair_fg(f, g, X, d, pref, rho);
            ris_boys<3>(rho * (X[0] * X[0] + X[1] * X[1] + X[2] * X[2]), boys3, F);
            const double m2r = -2.0 * rho;
            const double G[4] = {F[0], m2r * F[1], m2r * m2r * F[2], m2r * m2r * m2r * F[3]};
            const double w = (cf * dv[(size_t)s * n + q] + cv[(size_t)s * n + q] * df) * pref;
            for (int x = 0; x < 3; ++x) {
                d[nd] = x;
                acc[x] = fma(w, ris_dV(nd + 1, d, X, G), acc[x]);
            }
        }
    }
    __shared__ double red[3][128];
    for (int x = 0; x < 3; ++x) red[x][threadIdx.x] = acc[x];
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {
        if (threadIdx.x < o)
            for (int x = 0; x < 3; ++x) red[x][threadIdx.x] += red[x][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x < 3) grad[((size_t)s * gridDim.x + A) * 3 + threadIdx.x] = red[threadIdx.x][0];
}

extern "C" int ris_set_jfit(ris_ctx* c, int nshell_aux, const int32_t* aux_atom, const int32_t* aux_l, const double* aux_exp)
{
    if (!c || nshell_aux < 1 || !aux_atom || !aux_l || !aux_exp) return RIS_EINVAL;
    int nfn = 0;
    for (int i = 0; i < nshell_aux; ++i) {
        if (aux_atom[i] < 0 || aux_atom[i] >= c->natoms || aux_l[i] < 0 || aux_l[i] > 1 || !std::isfinite(aux_exp[i]) || !(aux_exp[i] > 0.0))
            return RIS_EINVAL;
        nfn += aux_l[i] ? 3 : 1;
    }
    CU(cudaSetDevice(c->device));
    std::vector<double> fn((size_t)RIS_AUX_FIELDS * nfn), lists[4];
    std::vector<int> lfn[4];
    std::vector<std::vector<int>> on_atom(c->natoms);
    int f = 0;
    for (int i = 0; i < nshell_aux; ++i)
        for (int comp = 0; comp < (aux_l[i] ? 3 : 1); ++comp, ++f) {
            double* r = &fn[(size_t)RIS_AUX_FIELDS * f];
            aux_record(r, &c->h_coords[3 * (size_t)aux_atom[i]], aux_exp[i], aux_l[i], comp, aux_atom[i], f);
            std::vector<double>& L = lists[aux_l[i] ? 1 + comp : 0];
            L.insert(L.end(), r, r + RIS_AUX_FIELDS);
            lfn[aux_l[i] ? 1 + comp : 0].push_back(f);
            on_atom[aux_atom[i]].push_back(f);
        }
    std::vector<int> off(c->natoms + 1, 0), idx;
    for (int a = 0; a < c->natoms; ++a) { idx.insert(idx.end(), on_atom[a].begin(), on_atom[a].end()); off[a + 1] = (int)idx.size(); }
    int rc;
    CU(cudaStreamSynchronize(c->stream));           // the host vectors below are read by async copies: finish them here
    if ((rc = dev_upload(c, &c->d_jfn, fn.data(), fn.size()))) return rc;
    for (int t = 0; t < 4; ++t) {
        c->jcnt[t] = (int)(lists[t].size() / RIS_AUX_FIELDS);
        c->h_jlist_fn[t] = lfn[t];
        c->d_jlist[t] = nullptr;
        if (c->jcnt[t] && (rc = dev_upload(c, &c->d_jlist[t], lists[t].data(), lists[t].size()))) return rc;
    }
    if ((rc = dev_upload(c, &c->d_atom_fn_off, off.data(), off.size()))) return rc;
    if ((rc = dev_upload(c, &c->d_atom_fn, idx.data(), idx.size()))) return rc;
    CU(cudaStreamSynchronize(c->stream));
    graphs_invalidate(c);
    c->jfit = true; c->naux_J = nfn; c->d_chol_J = nullptr; c->d_minv_J = nullptr;
    ris_resp_free(c);                       // stored Coulomb tensors belong to the previous set
    return RIS_OK;
}

extern "C" int ris_naux_J(const ris_ctx* c) { return c ? c->naux_J : RIS_EINVAL; }

// jset: the metric of the J-fit set (the default set when ris_set_jfit was never called)
static int metric_factor(ris_ctx* c, bool jset = false)
{
    const bool own = jset && c->jfit;
    double*& chol = own ? c->d_chol_J : c->d_chol;
    if (chol) return RIS_OK;
    const int n = own ? c->naux_J : c->naux;
    int rc;
    double* L;
    int* flag;
    if ((rc = dev_alloc(c, &L, (size_t)n * n, false))) return rc;
    if ((rc = dev_alloc(c, &flag, 1, true))) return rc;
    {
        ProfScope ps(c, "ris_k_metric", 40.0 * n * (double)n, 8.0 * n * (double)n);
        if (own) ris_k_metric_fn<<<(unsigned)(((long long)n * n + 255) / 256), 256, 0, c->stream>>>(n, c->d_jfn, c->d_boys[2], L);
        else ris_k_metric<<<(unsigned)(((long long)n * n + 255) / 256), 256, 0, c->stream>>>(n, c->d_aux, c->d_boys[0], L);
    }
    {
        ProfScope ps(c, "ris_k_cholesky", (double)n * n * n / 3.0, 8.0 * n * (double)n);
        ris_k_cholesky<<<1, 1024, 0, c->stream>>>(n, L, flag);
    }
    int hflag = 0;
    CU(cudaMemcpyAsync(&hflag, flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (hflag) return RIS_EINVAL;          // metric not positive definite (coincident aux centres)
    chol = L;
    return RIS_OK;
}

extern "C" int ris_metric_J(ris_ctx* c, double* M)
{
    if (!c || !M) return RIS_EINVAL;
    if (!c->jfit) return ris_metric(c, M);
    CU(cudaSetDevice(c->device));
    const int n = c->naux_J;
    ris_k_metric_fn<<<(unsigned)(((long long)n * n + 255) / 256), 256, 0, c->stream>>>(n, c->d_jfn, c->d_boys[2], M);
    CU(cudaGetLastError());
    return RIS_OK;
}

extern "C" int ris_metric(ris_ctx* c, double* M)
{
    if (!c || !M) return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    const int n = c->naux;
    ris_k_metric<<<(unsigned)(((long long)n * n + 255) / 256), 256, 0, c->stream>>>(n, c->d_aux, c->d_boys[0], M);
    CU(cudaGetLastError());
    return RIS_OK;
}

extern "C" int ris_fit_J(ris_ctx* c, int nbatch, const double* D, double* v_out, double* c_out)
{
    if (!c || nbatch < 1 || !D || !c_out) return RIS_EINVAL;
    if ((size_t)c->naux_J * sizeof(double) > 48 * 1024) return RIS_EINVAL;     // substitution vector in static-size shared memory
    CU(cudaSetDevice(c->device));
    int rc;
    if ((rc = metric_factor(c, true))) return rc;
    const long long nao2 = (long long)c->nao_in * c->nao_in;
    const int naux = c->naux_J;
    double* v = v_out;
    if (!v && (rc = ws_get(c, WS_OUT, sizeof(double) * (size_t)nbatch * naux, (void**)&v))) return rc;
    CU(cudaMemsetAsync(v, 0, sizeof(double) * (size_t)nbatch * naux, c->stream));
    for (int s0 = 0, nb; s0 < nbatch; s0 += nb) {
        nb = next_nb(nbatch - s0, RIS_NB_MAX);
        double* tile;
        if ((rc = ws_get(c, WS_TILE, sizeof(double) * (size_t)nb * c->nelem_real, (void**)&tile))) return rc;
        if ((rc = pack_tiles(c, D + (size_t)s0 * nao2, nao2, nb, tile, c->nelem_real))) return rc;
        for (int t = 0; t < 4; ++t) {       // one pass per type of auxiliary function: s, p_x, p_y, p_z
            const int nl = c->jcnt[t];
            if (nl == 0) continue;
            const int ny = (nl + 31) / 32;
            int* ctr;
            if ((rc = ws_get(c, WS_CTR, sizeof(int) * (size_t)2 * RIS_NCLASS * ny, (void**)&ctr))) return rc;
            CU(cudaMemsetAsync(ctr, 0, sizeof(int) * (size_t)2 * RIS_NCLASS * ny, c->stream));
            for (int oi = 0; oi < RIS_NCLASS; ++oi) {
                const int k = kClassOrder[oi];
                const RisClassPack& pk = c->cls[k];
                if (pk.npairs == 0) continue;
                RisGradParams p{};
                p.task_ctr = ctr + (size_t)2 * k * ny;
                p.pk = pk; p.naux = naux; p.natoms = c->natoms; p.nsm = c->nsm; p.aux = c->d_jlist[t]; p.aux_type = t;
                p.boys = c->d_boys[pk.la + pk.lb + (t ? 1 : 0)];
                p.tile = tile; p.sstride = c->nelem_real; p.estride = 1; p.lstride = 0; p.nb = nb;
                p.p0 = 0; p.p1 = nl; p.grad = v + (size_t)s0 * naux;
                const double nel = (double)ris_ncart(pk.la) * ris_ncart(pk.lb);
                ProfScope ps(c, kIntNames[k], (double)nl * ((double)pk.nprim * kModelFlopsByE[pk.la + pk.lb + (t ? 1 : 0)] + 2.0 * nel * pk.npairs * nb),
                             8.0 * nel * pk.npairs * nb + 8.0 * (double)pk.nprim * RIS_PRIM_FIELDS);
                CU(ris_int_launchers[k](p, c->stream));
            }
            CU(cudaGetLastError());
        }
    }
    {
        ProfScope ps(c, "ris_k_chol_solve", 2.0 * naux * (double)naux * nbatch, 8.0 * naux * (double)naux * nbatch);
        ris_k_chol_solve<<<nbatch, 256, sizeof(double) * naux, c->stream>>>(naux, c->jfit ? c->d_chol_J : c->d_chol, v, c_out);
    }
    CU(cudaGetLastError());
    return RIS_OK;
}

// --------------------------------------------------------------------------------------- fitting step, K type (NEXT-1)
//   T^P_ia = sum_{mu nu} C_occ[mu,i] (mu nu|P) C_vir[nu,a],   B = M^-1 T        (Eqs. 21-22)
// 1. ris_int_kernel<.., STORE>: the surviving (mu nu|P) into the P-minor integral buffer I[element][P]
// 2. ris_k_unpack_band: I -> per-P band slabs of the spatially ordered AO index: slab[P][row block][64][kw] (both
//    triangles; the band [jlo*64, jlo*64 + kw) of a row block covers every surviving partner of its rows)
// 3. GEMM-A (per row block, batched over P):  Ut[P][a][mu'] = sum_{nu' in band} C_vir^T[a][nu'] slab[P][mu'][nu']
// 4. GEMM-B (batched over P):                  T[P][i][a]   = sum_{mu'} C_occ^T[i][mu'] Ut[P][a][mu']
// 5. transpose T -> Tt[(i,a)][Q];  GEMM-C:     B[P][(i,a)]  = sum_Q Minv[P][Q] Tt[(i,a)][Q]
// all three GEMMs on the DMMA kernel of ris_gemm.cuh (K-contiguous "NT" operands).
__global__ void ris_k_unpack_band(RisClassPack pk, const int* __restrict__ ao_pos, int np, int pbp,
                                  const double* __restrict__ I, const int* __restrict__ rb_jlo, const int* __restrict__ rb_kw,
                                  const long long* __restrict__ rb_off, long long slab_stride, double* __restrict__ slab)
{
    const int nca = ris_ncart(pk.la), ncb = ris_ncart(pk.lb), nel = nca * ncb;
    const long long el = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (el >= (long long)nel * pk.npairs) return;
    const int P = blockIdx.y * 32 + (threadIdx.x & 31);
    if (P >= np) return;
    const int ip = (int)(el / nel), e = (int)(el - (long long)ip * nel);
    const int a0 = pk.ao[ip], b0 = pk.ao[(size_t)pk.npairs + ip];
    const int r = ao_pos[a0] + e / ncb, q = ao_pos[b0] + e % ncb;
    const double v = I[((size_t)pk.elem_off + (size_t)el) * pbp + P];
    double* s = slab + (size_t)P * slab_stride;
    {
        const int Ib = r / RIS_GTILE2;
        s[rb_off[Ib] + (long long)(r - Ib * RIS_GTILE2) * rb_kw[Ib] + (q - rb_jlo[Ib] * RIS_GTILE2)] = v;
    }
    if (a0 != b0) {          // a same-shell pair holds both (ca,cb) and (cb,ca) as elements of its own
        const int Ib = q / RIS_GTILE2;
        s[rb_off[Ib] + (long long)(q - Ib * RIS_GTILE2) * rb_kw[Ib] + (r - rb_jlo[Ib] * RIS_GTILE2)] = v;
    }
}

// out[col][pos] = in[order[pos]][col], pos < rows; zero for rows <= pos < ld   (C^T in spatial AO order, K-contiguous)
__global__ void ris_k_transpose_rows(int rows, int cols, int ld, const int* __restrict__ order, const double* __restrict__ in,
                                     double* __restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)cols * ld) return;
    const int col = (int)(i / ld), pos = (int)(i - (long long)col * ld);
    out[i] = pos < rows ? in[(size_t)order[pos] * cols + col] : 0.0;
}

// out[c][r] (ld ldo, zero padded) = in[r][c]: 32x32 tiles through shared memory
__global__ void ris_k_transpose(int rows, long long cols, int ldo, const double* __restrict__ in, double* __restrict__ out)
{
    __shared__ double t[32][33];
    const long long c0 = (long long)blockIdx.x * 32;
    const int r0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {
        const int r = r0 + j;
        const long long cc = c0 + threadIdx.x;
        t[j][threadIdx.x] = (r < rows && cc < cols) ? in[(size_t)r * cols + cc] : 0.0;
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {
        const long long cc = c0 + j;
        const int r = r0 + threadIdx.x;
        if (cc < cols && r < ldo) out[(size_t)cc * ldo + r] = t[threadIdx.x][j];
    }
}

__global__ void ris_k_eye(int n, double* __restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < (long long)n * n) out[i] = (i / n == i % n) ? 1.0 : 0.0;
}

__global__ void ris_k_pad2d(int rows, int cols, int ld, const double* __restrict__ in, double* __restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)rows * ld) return;
    const int r = (int)(i / ld), cidx = (int)(i - (long long)r * ld);
    out[i] = cidx < cols ? in[(size_t)r * cols + cidx] : 0.0;
}

static int metric_inverse(ris_ctx* c, bool jset = false)
{
    const bool own = jset && c->jfit;
    double*& slot = own ? c->d_minv_J : c->d_minv;
    if (slot) return RIS_OK;
    int rc;
    if ((rc = metric_factor(c, jset))) return rc;
    const int n = own ? c->naux_J : c->naux, np_ = (n + 1) & ~1;
    double *eye, *inv, *minv;
    if ((rc = dev_alloc(c, &eye, (size_t)n * n, false))) return rc;
    if ((rc = dev_alloc(c, &inv, (size_t)n * n, false))) return rc;
    if ((rc = dev_alloc(c, &minv, (size_t)n * np_, false))) return rc;
    const unsigned nb1 = (unsigned)(((long long)n * n + 255) / 256), nb2 = (unsigned)(((long long)n * np_ + 255) / 256);
    ris_k_eye<<<nb1, 256, 0, c->stream>>>(n, eye);
    ris_k_chol_solve<<<n, 256, sizeof(double) * n, c->stream>>>(n, own ? c->d_chol_J : c->d_chol, eye, inv);
    ris_k_pad2d<<<nb2, 256, 0, c->stream>>>(n, n, np_, inv, minv);
    CU(cudaGetLastError());
    slot = minv;
    return RIS_OK;
}

// The MO-basis three-index tensor over either auxiliary set, for any two coefficient matrices:
//   T[P][l][r] = sum_{mu nu} C_left[mu,l] (mu nu|P) C_right[nu,r]   (row length ldr >= nr, padding zero),  B = M^-1 T.
// jset: P runs over the J-fit set (its functions in input order) and M is its metric.  B_out may be null (no fit).
static int fit_mo(ris_ctx* c, bool jset, int nocc, int nvir, int ldr, const double* C_occ, const double* C_vir, double* T_out,
                  double* B_out)
{
    const bool own = jset && c->jfit;
    const int nao = c->nao, naux = own ? c->naux_J : c->naux;
    if ((size_t)naux * sizeof(double) > 48 * 1024 || ldr < nvir) return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    int rc;
    {   // spherical mode: Cartesian rows of the two coefficient matrices (one expansion when they are the same matrix)
        const bool same = C_occ == C_vir && nocc == nvir;
        if ((rc = sph_coef(c, WS_SPH_A, C_occ, nocc, &C_occ))) return rc;
        if (same) C_vir = C_occ;
        else if ((rc = sph_coef(c, WS_SPH_B, C_vir, nvir, &C_vir))) return rc;
    }
    if (B_out && (rc = metric_inverse(c, jset))) return rc;
    const int naop = (nao + 1) & ~1, nauxp = (naux + 1) & ~1, pbp = (naux + 3) & ~3;
    const long long nia = (long long)nocc * ldr;
    double *I, *slab, *Ut, *T, *Tt = nullptr, *CvT, *CoT;
    if ((rc = ws_get(c, WS_FIT_I, sizeof(double) * (size_t)std::max<long long>(c->nelem_real, 1) * pbp, (void**)&I))) return rc;
    if ((rc = ws_get(c, WS_FIT_SLAB, sizeof(double) * (size_t)naux * c->slab_stride, (void**)&slab))) return rc;
    if ((rc = ws_get(c, WS_FIT_UT, sizeof(double) * (size_t)naux * nvir * naop, (void**)&Ut))) return rc;
    if (B_out && (rc = ws_get(c, WS_FIT_TT, sizeof(double) * (size_t)nia * nauxp, (void**)&Tt))) return rc;
    if ((rc = ws_get(c, WS_FIT_CV, sizeof(double) * (size_t)nvir * naop, (void**)&CvT))) return rc;
    if ((rc = ws_get(c, WS_FIT_CO, sizeof(double) * (size_t)nocc * naop, (void**)&CoT))) return rc;
    T = T_out;
    if (!T && (rc = ws_get(c, WS_FIT_T, sizeof(double) * (size_t)naux * nia, (void**)&T))) return rc;
    CU(cudaMemsetAsync(I, 0, sizeof(double) * (size_t)std::max<long long>(c->nelem_real, 1) * pbp, c->stream));
    CU(cudaMemsetAsync(slab, 0, sizeof(double) * (size_t)naux * c->slab_stride, c->stream));
    if (ldr != nvir) CU(cudaMemsetAsync(T, 0, sizeof(double) * (size_t)naux * nia, c->stream));
    const int ny = (naux + 31) / 32;
    for (int t = 0; t < (own ? 4 : 1); ++t) {   // 1. integrals, one pass per type of auxiliary function
        const int nl = own ? c->jcnt[t] : naux;
        if (nl == 0) continue;
        const int nyl = (nl + 31) / 32;
        int* ctr;
        if ((rc = ws_get(c, WS_CTR, sizeof(int) * (size_t)2 * RIS_NCLASS * nyl, (void**)&ctr))) return rc;
        CU(cudaMemsetAsync(ctr, 0, sizeof(int) * (size_t)2 * RIS_NCLASS * nyl, c->stream));
        for (int oi = 0; oi < RIS_NCLASS; ++oi) {
            const int k = kClassOrder[oi];
            const RisClassPack& pk = c->cls[k];
            if (pk.npairs == 0) continue;
            RisGradParams p{};
            p.task_ctr = ctr + (size_t)2 * k * nyl;
            p.pk = pk; p.naux = naux; p.natoms = c->natoms; p.nsm = c->nsm; p.aux = own ? c->d_jlist[t] : c->d_aux; p.aux_type = t;
            p.boys = c->d_boys[pk.la + pk.lb + (t ? 1 : 0)];
            p.estride = pbp; p.nb = 0; p.p0 = 0; p.p1 = nl; p.grad = I;
            const double nel = (double)ris_ncart(pk.la) * ris_ncart(pk.lb);
            ProfScope ps(c, kIntNames[k], (double)nl * (double)pk.nprim * kModelFlopsByE[pk.la + pk.lb + (t ? 1 : 0)],
                         8.0 * nel * pk.npairs * nl + 8.0 * (double)pk.nprim * RIS_PRIM_FIELDS);
            CU(ris_ints_launchers[k](p, c->stream));
        }
        CU(cudaGetLastError());
    }
    {   // 2. band slabs
        ProfScope ps(c, "ris_k_unpack_band", 0.0, 24.0 * (double)c->nelem_real * naux);
        for (int k = 0; k < RIS_NCLASS; ++k) {
            const RisClassPack& pk = c->cls[k];
            if (pk.npairs == 0) continue;
            const long long nelc = (long long)ris_ncart(pk.la) * ris_ncart(pk.lb) * pk.npairs;
            ris_k_unpack_band<<<dim3((unsigned)((nelc + 7) / 8), ny), 256, 0, c->stream>>>(pk, c->d_ao_pos, naux, pbp, I, c->d_rb_jlo,
                                                                                         c->d_rb_kw, c->d_rb_off, c->slab_stride, slab);
        }
        CU(cudaGetLastError());
    }
    {
        const long long n1 = (long long)nvir * naop, n2 = (long long)nocc * naop;
        ris_k_transpose_rows<<<(unsigned)((n1 + 255) / 256), 256, 0, c->stream>>>(nao, nvir, naop, c->d_ao_order, C_vir, CvT);
        ris_k_transpose_rows<<<(unsigned)((n2 + 255) / 256), 256, 0, c->stream>>>(nao, nocc, naop, c->d_ao_order, C_occ, CoT);
        CU(cudaGetLastError());
    }
    double flopsA = 0.0;
    for (int Ib = 0; Ib < c->nblk; ++Ib) flopsA += 2.0 * naux * (double)nvir * std::min(RIS_GTILE2, nao - Ib * RIS_GTILE2) * c->rb_kw[Ib];
    {   // 3. GEMM-A, one launch per row block, batched over P
        ProfScope ps(c, "ris_gemm_dmma(Ut=CvirT*slab^T,band)", flopsA, 8.0 * ((double)naux * c->slab_stride + (double)naux * nvir * nao));
        for (int Ib = 0; Ib < c->nblk; ++Ib) {
            const int col0 = c->rb_jlo[Ib] * RIS_GTILE2;
            RisGemmParams g{};
            g.seg[0] = RisGemmSeg{CvT + col0, naop, 0, slab + c->rb_off[Ib], c->rb_kw[Ib], c->slab_stride,
                                  std::min(c->rb_kw[Ib], naop - col0)};
            g.nseg = 1; g.M = nvir; g.N = std::min(RIS_GTILE2, nao - Ib * RIS_GTILE2);
            g.C = Ut + (size_t)Ib * RIS_GTILE2; g.ldc = naop; g.bsC = (long long)nvir * naop;
            CU((ris_gemm_launch_cfg<RIS_GTILE2, RIS_GTILE2, 32, 32, 3, 3>(c->stream, g, naux, 0)));
        }
    }
    {   // 4. GEMM-B: T[P][i][a]
        RisGemmParams g{};
        g.seg[0] = RisGemmSeg{CoT, naop, 0, Ut, naop, (long long)nvir * naop, nao};
        g.nseg = 1; g.M = nocc; g.N = nvir; g.C = T; g.ldc = ldr; g.bsC = nia;
        ProfScope ps(c, "ris_gemm_dmma(T=CoccT*Ut^T)", 2.0 * naux * (double)nocc * nvir * nao,
                     8.0 * ((double)naux * nvir * nao + (double)naux * nia));
        CU(ris_gemm_dense(c->stream, g, naux));
    }
    if (!B_out) return RIS_OK;
    {   // 5. Tt[(i,a)][Q], then B[P][(i,a)] = sum_Q Minv[P][Q] Tt[(i,a)][Q]
        ProfScope ps(c, "ris_k_transpose", 0.0, 16.0 * naux * (double)nia);
        ris_k_transpose<<<dim3((unsigned)((nia + 31) / 32), (nauxp + 31) / 32), dim3(32, 8), 0, c->stream>>>(naux, nia, nauxp, T, Tt);
        CU(cudaGetLastError());
    }
    {
        RisGemmParams g{};
        g.seg[0] = RisGemmSeg{Tt, nauxp, 0, own ? c->d_minv_J : c->d_minv, nauxp, 0, naux};
        g.nseg = 1; g.M = (int)nia; g.N = naux; g.C = B_out; g.ldc = 1; g.bsC = 0;
        g.cdiv = 1; g.cpad = nia;
        ProfScope ps(c, "ris_gemm_dmma(B=Minv*T)", 2.0 * naux * (double)naux * nia, 16.0 * naux * (double)nia);
        CU(ris_gemm_dense(c->stream, g, 1));
    }
    return RIS_OK;
}

extern "C" int ris_fit_K(ris_ctx* c, int nocc, int nvir, const double* C_occ, const double* C_vir, double* T_out, double* B_out)
{
    if (!c || nocc < 1 || nvir < 1 || !C_occ || !C_vir || !B_out) return RIS_EINVAL;
    return fit_mo(c, false, nocc, nvir, nvir, C_occ, C_vir, T_out, B_out);
}

#include "ris_resp.cuh"

// Metric term of Eq. 27 with a FULL matrix: g[s][A] = sum_{PQ} G[s][P][Q] d(P|Q)/dR_A, positive sign.
__global__ void __launch_bounds__(128) ris_k_grad_pq_full(int naux, const double* __restrict__ aux, const double* __restrict__ boys1,
                                                          const double* __restrict__ G, double* __restrict__ grad)
{
    const int P = blockIdx.x, s = blockIdx.y;
    const double* Gs = G + (size_t)s * naux * naux;
    const double Px = aux[RIS_AUX_FIELDS * P], Py = aux[RIS_AUX_FIELDS * P + 1], Pz = aux[RIS_AUX_FIELDS * P + 2], al = aux[RIS_AUX_FIELDS * P + 3], fP = aux[RIS_AUX_FIELDS * P + 4];
    double g0 = 0.0, g1 = 0.0, g2 = 0.0;
    for (int Q = threadIdx.x; Q < naux; Q += blockDim.x) {
        if (Q == P) continue;
        const double X0 = Px - aux[RIS_AUX_FIELDS * Q], X1 = Py - aux[RIS_AUX_FIELDS * Q + 1], X2 = Pz - aux[RIS_AUX_FIELDS * Q + 2];
        const double be = aux[RIS_AUX_FIELDS * Q + 3], fQ = aux[RIS_AUX_FIELDS * Q + 4];
        const double sI = ris_rsqrt(al + be);
        const double rho = al * be * sI * sI;
        double F[2];
        ris_boys<1>(rho * (X0 * X0 + X1 * X1 + X2 * X2), boys1, F);
        const double w = (Gs[(size_t)P * naux + Q] + Gs[(size_t)Q * naux + P]) * fP * fQ * (2.0 * 17.493418327624862846) * sI *
                         (-2.0 * rho) * F[1];
        g0 = fma(w, X0, g0); g1 = fma(w, X1, g1); g2 = fma(w, X2, g2);
    }
    __shared__ double red[3][128];
    red[0][threadIdx.x] = g0; red[1][threadIdx.x] = g1; red[2][threadIdx.x] = g2;
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {
        if (threadIdx.x < o)
            for (int x = 0; x < 3; ++x) red[x][threadIdx.x] += red[x][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x < 3) grad[((size_t)s * naux + P) * 3 + threadIdx.x] = red[threadIdx.x][0];
}

extern "C" int ris_grad_PQ_full(ris_ctx* c, int nbatch, const double* G, double* grad)
{
    if (!c || nbatch < 1 || !G || !grad) return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    ProfScope ps(c, "ris_k_grad_pq_full", 60.0 * c->naux * (double)c->naux * nbatch, 8.0 * c->naux * (double)c->naux * nbatch);
    ris_k_grad_pq_full<<<dim3(c->naux, nbatch), 128, 0, c->stream>>>(c->naux, c->d_aux, c->d_boys[1], G, grad);
    CU(cudaGetLastError());
    return RIS_OK;
}

// --------------------------------------------------------------------------------------- K
// out[pos][0..ld) = in[order[pos]][0..cols) zero padded: C_occ in spatial row order with an even leading dimension
__global__ void ris_k_pad_rows(int rows, int cols, int ld, const int* __restrict__ order, const double* __restrict__ in,
                               double* __restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)rows * ld) return;
    const int r = (int)(i / ld), cidx = (int)(i - (long long)r * ld);
    out[i] = cidx < cols ? in[(size_t)order[r] * cols + cidx] : 0.0;
}

// b_ready (nullable): b_ready[s * RIS_COPY_CHUNKS + ch] is recorded (on another stream) once chunk ch (a range of P) of
// B of state s is resident; the compute stream waits for it right before that chunk's GEMM-1, so the H2D copy runs
// ahead of the GEMMs instead of in front of them.
constexpr int RIS_COPY_CHUNKS = 8;     // *_host: B of a state goes up in this many P ranges, GEMM-1 follows chunk by chunk
// [p_lo, p_hi): the aux functions this call sums over (all of them, or one rank's share when the K term is sharded over P);
// B then holds only those: [nbatch][p_hi - p_lo][nocc][nvir].
static int grad_K_impl(ris_ctx* c, int nbatch, int nocc, int nvir, const double* C_occ, const double* C_vir,
                       const double* B, double* grad, const cudaEvent_t* b_ready, int p_lo = 0, int p_hi = -1)
{
    if (!c || nbatch < 1 || nocc < 1 || nvir < 1 || !C_occ || !C_vir || !grad) return RIS_EINVAL;
    if (p_hi < 0) p_hi = c->naux;
    if (p_lo < 0 || p_hi > c->naux || p_lo > p_hi) return RIS_EINVAL;
    const int nloc = p_hi - p_lo;
    if (!B && nloc > 0) return RIS_EINVAL;              // an empty share has no B
    CU(cudaSetDevice(c->device));
    CU(cudaMemsetAsync(grad, 0, sizeof(double) * (size_t)nbatch * c->natoms * 3, c->stream));
    if (c->nelem_real == 0 || nloc == 0) return RIS_OK;   // every shell pair screened out / empty share: exactly zero
    const int nao = c->nao, naux = nloc;
    { int rc0; if ((rc0 = sph_coef(c, WS_SPH_A, C_occ, nocc, &C_occ)) || (rc0 = sph_coef(c, WS_SPH_B, C_vir, nvir, &C_vir))) return rc0; }
    const int cap = nb_cap(c, true);
    if (cap < 1) return RIS_ENOMEM;
    const int nbmax = next_nb(nbatch, cap);
    const int noccp = (nocc + 1) & ~1;                    // even: 16-byte aligned sub-blocks of HT
    // per aux function: HT [nao][noccp], packed tiles [nb][elements]
    int pb = c->opt.p_batch;
    if (pb <= 0) {
        size_t fr = 0, tot = 0;
        CU(cudaMemGetInfo(&fr, &tot));
        fr += c->ws_bytes[WS_TILE] + c->ws_bytes[WS_H];
        const double per = 8.0 * ((double)noccp * nao + (double)nbmax * c->nelem_real);
        const double budget = std::min(0.5 * (double)fr, 24.0e9);
        pb = (int)std::max(1.0, std::min((double)naux, budget / per));
        if (pb < naux && pb > 32) pb &= ~31;              // whole chunks of 32 aux lanes
    }
    pb = std::min(pb, naux);
    c->last_pbatch = pb;
    const int pbp = (pb + 3) & ~3;                        // P-minor tile rows start on 32-byte sectors
    double *tile, *HT, *Cop;
    int rc;
    unsigned long long* det;
    if ((rc = det_begin(c, nbatch, &det))) return rc;
    if ((rc = ws_get(c, WS_TILE, sizeof(double) * (size_t)nbmax * pbp * c->nelem_real, (void**)&tile))) return rc;
    if ((rc = ws_get(c, WS_H, sizeof(double) * (size_t)nao * pb * noccp, (void**)&HT))) return rc;
    if ((rc = ws_get(c, WS_COCC, sizeof(double) * (size_t)nao * noccp, (void**)&Cop))) return rc;
    {
        ProfScope ps(c, "ris_k_pad_rows", 0.0, 16.0 * nao * (double)noccp);
        const long long n = (long long)nao * noccp;
        ris_k_pad_rows<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(nao, nocc, noccp, c->d_ao_order, C_occ, Cop);
    }
    for (int s0 = 0, nb; s0 < nbatch; s0 += nb) {
        nb = next_nb(nbatch - s0, cap);
        for (int p0 = 0; p0 < naux; p0 += pb) {
            const int np = std::min(pb, naux - p0);
            const long long ldh = (long long)pb * noccp;
            {   // the GEMM-2 epilogue ADDS the two halves of every element
                ProfScope ps(c, "memset(K tiles)", 0.0, 8.0 * nb * (double)pbp * c->nelem_real);
                CU(cudaMemsetAsync(tile, 0, sizeof(double) * (size_t)nb * pbp * c->nelem_real, c->stream));
            }
            for (int s = 0; s < nb; ++s) {
                const double* Bs = B + (((size_t)(s0 + s) * naux + p0) * nocc) * nvir;      // p0: offset within the share
                // GEMM-1: HT[nu][(P,i)] = sum_a C_vir[nu][a] B[P][i][a]; with b_ready, in RIS_COPY_CHUNKS column chunks
                // (ranges of P), each waiting only for its own slice of B
                const int nch = (b_ready && p0 == 0 && np == naux) ? RIS_COPY_CHUNKS : 1;
                for (int ch = 0; ch < nch; ++ch) {
                    const int q0 = (int)((long long)np * ch / nch), q1 = (int)((long long)np * (ch + 1) / nch);
                    if (q1 <= q0) continue;
                    if (b_ready) {
                        if (nch > 1) CU(cudaStreamWaitEvent(c->stream, b_ready[(s0 + s) * RIS_COPY_CHUNKS + ch], 0));
                        else if (p0 == 0) CU(cudaStreamWaitEvent(c->stream, b_ready[(s0 + s) * RIS_COPY_CHUNKS + RIS_COPY_CHUNKS - 1], 0));
                    }
                    RisGemmParams g{};
                    g.seg[0] = RisGemmSeg{C_vir, nvir, 0, Bs + (size_t)q0 * nocc * nvir, nvir, 0, nvir};
                    g.nseg = 1; g.M = nao; g.N = (q1 - q0) * nocc; g.C = HT + (size_t)q0 * noccp; g.ldc = ldh; g.bsC = 0;
                    g.rowsA = c->d_ao_order;                  // HT rows in spatial order
                    g.cdiv = (noccp != nocc) ? nocc : 0; g.cpad = noccp;
                    ProfScope ps(c, "ris_gemm_dmma(HT=Cvir*B^T)", 2.0 * (q1 - q0) * nocc * (double)nao * nvir,
                                 8.0 * ((double)(q1 - q0) * nocc * nvir + (double)nao * nvir + (double)(q1 - q0) * nocc * nao));
                    CU(ris_gemm_dense(c->stream, g, 1));
                }
                {   // GEMM-2: tile[e][P] += f Gamma^P_{mu nu}, one column problem per AO, P as the N dimension (scatter mode)
                    double* out = tile + (size_t)s * pbp * c->nelem_real;
                    RisGemmParams g{};
                    g.seg[0] = RisGemmSeg{Cop, noccp, 0, HT, noccp, ldh, nocc};
                    g.nseg = 1; g.M = nao; g.N = np; g.C = out; g.ldc = pbp; g.bsC = 0;
                    g.tiles = c->d_g2tiles; g.srows = c->d_g2rows; g.scode = c->d_g2code;
                    // algorithmic flops: two length-nocc dot products per unique surviving pair element
                    ProfScope ps(c, "ris_gemm_dmma(tile+=Cocc*HT^T,scatter)", 4.0 * np * nocc * (double)c->nelem_real,
                                 8.0 * np * ((double)noccp * nao + 3.0 * (double)c->nelem_real) + 8.0 * nao * noccp);
                    CU(ris_gemm_scatter(c->stream, g, c->ntiles));
                }
            }
            if ((rc = launch_classes(c, tile, (long long)pbp * c->nelem_real, pbp, 1, nullptr, nb, p_lo + p0, p_lo + p0 + np,
                                     grad + (size_t)s0 * c->natoms * 3, det ? det + (size_t)2 * s0 * c->natoms * 3 : nullptr)))
                return rc;
        }
    }
    return det_end(c, nbatch, det, grad);
}

static int grad_K_graphed(ris_ctx* c, int nbatch, int nocc, int nvir, const double* C_occ, const double* C_vir, const double* B,
                          double* grad, int p_lo, int p_hi)
{
    const std::vector<unsigned long long> key = {2ull, (unsigned long long)nbatch, (unsigned long long)nocc, (unsigned long long)nvir,
                                                 key_of(C_occ), key_of(C_vir), key_of(B), key_of(grad),
                                                 (unsigned long long)(long long)p_lo, (unsigned long long)(long long)p_hi};
    return run_graphed(c, 1, key, [&]() { return grad_K_impl(c, nbatch, nocc, nvir, C_occ, C_vir, B, grad, nullptr, p_lo, p_hi); });
}
extern "C" int ris_grad_K(ris_ctx* c, int nbatch, int nocc, int nvir, const double* C_occ, const double* C_vir,
                          const double* B, double* grad)
{
    if (!c) return RIS_EINVAL;
    return grad_K_graphed(c, nbatch, nocc, nvir, C_occ, C_vir, B, grad, 0, -1);
}

extern "C" int ris_grad_K_range(ris_ctx* c, int nbatch, int nocc, int nvir, const double* C_occ, const double* C_vir,
                                const double* B_local, int p_lo, int p_hi, double* grad)
{
    if (!c || p_lo < 0 || p_hi < p_lo) return RIS_EINVAL;
    return grad_K_graphed(c, nbatch, nocc, nvir, C_occ, C_vir, B_local, grad, p_lo, p_hi);
}

// --------------------------------------------------------------------------------------- PQ (S5)
// g[s][P] = sum_{Q != P} (c_P d_Q + c_Q d_P) N_P N_Q d(P|Q)/dR_P,
// d(P|Q)/dR_P = -2 rho (R_P - R_Q) 2 pi^{5/2}/(alpha beta sqrt(alpha+beta)) F_1(rho R^2)   (Eq. 22).
// One block per aux P, threads over Q, fixed-order block reduction: deterministic, no atomics.
__global__ void __launch_bounds__(128) ris_k_grad_pq(int naux, int nb, const double* __restrict__ aux,
                                                     const double* __restrict__ boys1, const double* __restrict__ cv,
                                                     const double* __restrict__ dv, double* __restrict__ grad)
{
    const int P = blockIdx.x, s = blockIdx.y;
    const double Px = aux[RIS_AUX_FIELDS * P], Py = aux[RIS_AUX_FIELDS * P + 1], Pz = aux[RIS_AUX_FIELDS * P + 2], al = aux[RIS_AUX_FIELDS * P + 3], fP = aux[RIS_AUX_FIELDS * P + 4];
    const double cP = cv[(size_t)s * naux + P], dP = dv[(size_t)s * naux + P];
    double g0 = 0.0, g1 = 0.0, g2 = 0.0;
    for (int Q = threadIdx.x; Q < naux; Q += blockDim.x) {
        if (Q == P) continue;
        const double X0 = Px - aux[RIS_AUX_FIELDS * Q], X1 = Py - aux[RIS_AUX_FIELDS * Q + 1], X2 = Pz - aux[RIS_AUX_FIELDS * Q + 2];
        const double be = aux[RIS_AUX_FIELDS * Q + 3], fQ = aux[RIS_AUX_FIELDS * Q + 4];
        const double sI = ris_rsqrt(al + be);
        const double rho = al * be * sI * sI;
        double F[2];
        ris_boys<1>(rho * (X0 * X0 + X1 * X1 + X2 * X2), boys1, F);
        // N_P N_Q/(alpha beta) = fP fQ
        const double w = (cP * dv[(size_t)s * naux + Q] + cv[(size_t)s * naux + Q] * dP) * fP * fQ *
                         (2.0 * 17.493418327624862846) * sI * (-2.0 * rho) * F[1];
        g0 = fma(w, X0, g0); g1 = fma(w, X1, g1); g2 = fma(w, X2, g2);
    }
    __shared__ double red[3][128];
    red[0][threadIdx.x] = g0; red[1][threadIdx.x] = g1; red[2][threadIdx.x] = g2;
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {
        if (threadIdx.x < o)
            for (int x = 0; x < 3; ++x) red[x][threadIdx.x] += red[x][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x < 3) grad[((size_t)s * naux + P) * 3 + threadIdx.x] = red[threadIdx.x][0];
}

extern "C" int ris_grad_PQ(ris_ctx* c, int nbatch, const double* c_aux, const double* d_aux, double* grad)
{
    if (!c || nbatch < 1 || !c_aux || !d_aux || !grad) return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    ProfScope ps(c, "ris_k_grad_pq", 60.0 * c->naux_J * (double)c->naux_J * nbatch, 0.0);
    if (c->jfit)
        ris_k_grad_pq_fn<<<dim3(c->natoms, nbatch), 128, 0, c->stream>>>(c->naux_J, c->d_jfn, c->d_atom_fn_off, c->d_atom_fn, c->d_boys[3],
                                                                       c_aux, d_aux, grad);
    else
        ris_k_grad_pq<<<dim3(c->naux, nbatch), 128, 0, c->stream>>>(c->naux, nbatch, c->d_aux, c->d_boys[1], c_aux, d_aux, grad);
    CU(cudaGetLastError());
    return RIS_OK;
}

// --------------------------------------------------------------------------------------- host-buffer entry points
static int h2d(ris_ctx* c, int slot, const double* h, size_t n, double** d)
{
    int rc = ws_get(c, slot, n * sizeof(double), (void**)d);
    if (rc) return rc;
    CU(cudaMemcpyAsync(*d, h, n * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    return RIS_OK;
}

static int d2h_grad(ris_ctx* c, const double* d, double* h, size_t n)
{
    CU(cudaMemcpyAsync(h, d, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return RIS_OK;
}

extern "C" int ris_grad_J_host(ris_ctx* c, int nbatch, const double* D, const double* c_aux, double* grad)
{
    if (!c || nbatch < 1 || !D || !c_aux || !grad) return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    double *dD, *dc, *dg;
    int rc;
    const size_t ng = (size_t)nbatch * c->natoms * 3;
    if ((rc = h2d(c, WS_IN0, D, (size_t)nbatch * c->nao_in * c->nao_in, &dD))) return rc;
    if ((rc = h2d(c, WS_IN1, c_aux, (size_t)nbatch * c->naux_J, &dc))) return rc;
    if ((rc = ws_get(c, WS_OUT, ng * sizeof(double), (void**)&dg))) return rc;
    if ((rc = ris_grad_J(c, nbatch, dD, dc, dg))) return rc;
    return d2h_grad(c, dg, grad, ng);
}

// B [nbatch][naux][nocc][nvir] host -> device staging (WS_IN0) on the copy stream, in RIS_COPY_CHUNKS ranges of P per state,
// one event per chunk (c->copy_ev[s * RIS_COPY_CHUNKS + ch]).  The caller has already enqueued the small operands: the
// H2D copy engine serves transfers in issue order across streams.
static int upload_B_chunked(ris_ctx* c, int nbatch, int nocc, int nvir, const double* B, double** dB_out,
                            const double* extra_h = nullptr, double* extra_d = nullptr, size_t extra_n = 0)
{
    int rc;
    double* dB;
    const size_t nB = (size_t)c->naux * nocc * nvir;
    if ((rc = ws_get(c, WS_IN0, nbatch * nB * sizeof(double), (void**)&dB))) return rc;
    if (!c->copy_stream) CU(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    if (!c->copy_gate) CU(cudaEventCreateWithFlags(&c->copy_gate, cudaEventDisableTiming));
    while ((int)c->copy_ev.size() < nbatch * RIS_COPY_CHUNKS) {
        cudaEvent_t e;
        CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        c->copy_ev.push_back(e);
    }
    CU(cudaEventRecord(c->copy_gate, c->stream));                 // earlier readers of the staging buffer are done
    CU(cudaStreamWaitEvent(c->copy_stream, c->copy_gate, 0));
    for (int s = 0; s < nbatch; ++s)
        for (int ch = 0; ch < RIS_COPY_CHUNKS; ++ch) {
            const size_t q0 = (size_t)((long long)c->naux * ch / RIS_COPY_CHUNKS) * nocc * nvir;
            const size_t q1 = (size_t)((long long)c->naux * (ch + 1) / RIS_COPY_CHUNKS) * nocc * nvir;
            if (q1 > q0)
                CU(cudaMemcpyAsync(dB + s * nB + q0, B + s * nB + q0, (q1 - q0) * sizeof(double), cudaMemcpyHostToDevice, c->copy_stream));
            CU(cudaEventRecord(c->copy_ev[s * RIS_COPY_CHUNKS + ch], c->copy_stream));
            if (s == 0 && ch == RIS_COPY_CHUNKS - 1 && extra_n > 0) {
                // a second payload (D of the combined call) rides behind the first state's B: its consumer runs last
                if (!c->copy_extra) CU(cudaEventCreateWithFlags(&c->copy_extra, cudaEventDisableTiming));
                CU(cudaMemcpyAsync(extra_d, extra_h, extra_n * sizeof(double), cudaMemcpyHostToDevice, c->copy_stream));
                CU(cudaEventRecord(c->copy_extra, c->copy_stream));
            }
        }
    *dB_out = dB;
    return RIS_OK;
}

extern "C" int ris_grad_K_host(ris_ctx* c, int nbatch, int nocc, int nvir, const double* C_occ, const double* C_vir,
                               const double* B, double* grad)
{
    if (!c || nbatch < 1 || nocc < 1 || nvir < 1 || !C_occ || !C_vir || !B || !grad) return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    double *dCo, *dCv, *dB, *dg;
    int rc;
    const size_t ng = (size_t)nbatch * c->natoms * 3;
    // B (the bulk of the input: naux*nocc*nvir doubles per state) goes up state by state on a second stream, each
    // state's GEMMs waiting only for their own slice: the PCIe transfer of state s+1 hides behind the GEMMs of state s.
    // The small operands go first: the H2D copy engine serves transfers in issue order across streams.
    if ((rc = h2d(c, WS_IN1, C_occ, (size_t)c->nao_in * nocc, &dCo))) return rc;
    if ((rc = h2d(c, WS_IN2, C_vir, (size_t)c->nao_in * nvir, &dCv))) return rc;
    if ((rc = upload_B_chunked(c, nbatch, nocc, nvir, B, &dB))) return rc;
    if ((rc = ws_get(c, WS_OUT, ng * sizeof(double), (void**)&dg))) return rc;
    if ((rc = grad_K_impl(c, nbatch, nocc, nvir, dCo, dCv, dB, dg, c->copy_ev.data()))) {
        cudaStreamSynchronize(c->copy_stream);
        return rc;
    }
    return d2h_grad(c, dg, grad, ng);
}

extern "C" int ris_grad_PQ_host(ris_ctx* c, int nbatch, const double* c_aux, const double* d_aux, double* grad)
{
    if (!c || nbatch < 1 || !c_aux || !d_aux || !grad) return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    double *dc, *dd, *dg;
    int rc;
    const size_t ng = (size_t)nbatch * c->natoms * 3;
    if ((rc = h2d(c, WS_IN0, c_aux, (size_t)nbatch * c->naux_J, &dc))) return rc;
    if ((rc = h2d(c, WS_IN1, d_aux, (size_t)nbatch * c->naux_J, &dd))) return rc;
    if ((rc = ws_get(c, WS_OUT, ng * sizeof(double), (void**)&dg))) return rc;
    if ((rc = ris_grad_PQ(c, nbatch, dc, dd, dg))) return rc;
    return d2h_grad(c, dg, grad, ng);
}

// All three terms on host buffers in ONE call: the chunked upload of B starts right behind the small operands and D,
// so it runs under the J class kernels and the GEMMs of the chunks already resident; one synchronisation at the end.
extern "C" int ris_grad_host(ris_ctx* c, int nbJ, const double* D, const double* c_aux, const double* d_aux, int nbK, int nocc,
                             int nvir, const double* C_occ, const double* C_vir, const double* B, double* grad_J, double* grad_K,
                             double* grad_PQ)
{
    if (!c || nbJ < 1 || nbK < 1 || nocc < 1 || nvir < 1 || !D || !c_aux || !d_aux || !C_occ || !C_vir || !B || !grad_J || !grad_K ||
        !grad_PQ)
        return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    int rc;
    double *dc, *dd, *dCo, *dCv, *dD, *dB, *dg;
    const size_t nJ = (size_t)nbJ * c->natoms * 3, nK = (size_t)nbK * c->natoms * 3;
    if ((rc = h2d(c, WS_HC, c_aux, (size_t)nbJ * c->naux_J, &dc))) return rc;
    if ((rc = h2d(c, WS_HDQ, d_aux, (size_t)nbJ * c->naux_J, &dd))) return rc;
    if ((rc = h2d(c, WS_IN1, C_occ, (size_t)c->nao_in * nocc, &dCo))) return rc;
    if ((rc = h2d(c, WS_IN2, C_vir, (size_t)c->nao_in * nvir, &dCv))) return rc;
    const size_t nD = (size_t)nbJ * c->nao_in * c->nao_in;
    if ((rc = ws_get(c, WS_HD, nD * sizeof(double), (void**)&dD))) return rc;
    if ((rc = upload_B_chunked(c, nbK, nocc, nvir, B, &dB, D, dD, nD))) return rc;
    if ((rc = ws_get(c, WS_OUT, (2 * nJ + nK) * sizeof(double), (void**)&dg))) return rc;
    // compute order: PQ (needs only c, d), K (follows the chunks of B), J last (D rode up behind the first state's B)
    if ((rc = ris_grad_PQ(c, nbJ, dc, dd, dg + nJ)) ||
        (rc = grad_K_impl(c, nbK, nocc, nvir, dCo, dCv, dB, dg + 2 * nJ, c->copy_ev.data()))) {
        cudaStreamSynchronize(c->copy_stream);
        return rc;
    }
    CU(cudaStreamWaitEvent(c->stream, c->copy_extra, 0));
    if ((rc = ris_grad_J(c, nbJ, dD, dc, dg))) { cudaStreamSynchronize(c->copy_stream); return rc; }
    CU(cudaMemcpyAsync(grad_J, dg, nJ * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaMemcpyAsync(grad_PQ, dg + nJ, nJ * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaMemcpyAsync(grad_K, dg + 2 * nJ, nK * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return RIS_OK;
}

// --------------------------------------------------------------------------------------- FP64 probe
__global__ void ris_k_dfma_probe(double* out, int iters, double a, double b)
{
    double x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    if (s == 12345.678) out[0] = s;
}

__global__ void ris_k_dmma_probe(double* out, int iters)
{
    double c0[2] = {0, 0}, c1[2] = {0, 0}, c2[2] = {0, 0}, c3[2] = {0, 0};
    const double a = threadIdx.x * 1e-3, b = 1.0 + threadIdx.x * 1e-4;
    for (int it = 0; it < iters; ++it) {
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};" : "+d"(c0[0]), "+d"(c0[1]) : "d"(a), "d"(b));
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};" : "+d"(c1[0]), "+d"(c1[1]) : "d"(a), "d"(b));
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};" : "+d"(c2[0]), "+d"(c2[1]) : "d"(a), "d"(b));
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};" : "+d"(c3[0]), "+d"(c3[1]) : "d"(a), "d"(b));
    }
    const double s = c0[0] + c0[1] + c1[0] + c1[1] + c2[0] + c2[1] + c3[0] + c3[1];
    if (s == 12345.678) out[0] = s;
}

// kind 0: independent DFMA chains (FP64 FMA pipe); kind 1: mma.sync m8n8k4 f64 chains (FP64 tensor path)
static int probe_fp64(int kind, double* tflops, void* cuda_stream)
{
    if (!tflops) return RIS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, nsm = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    double* d;
    CU(cudaMalloc(&d, 8));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    const int iters = 40000, thr = 512;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        CU(cudaEventRecord(e0, st));
        if (kind == 0) ris_k_dfma_probe<<<nsm, thr, 0, st>>>(d, iters, 1.0000001, 1e-9);
        else ris_k_dmma_probe<<<nsm, thr, 0, st>>>(d, iters);
        CU(cudaEventRecord(e1, st));
        CU(cudaEventSynchronize(e1));
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, e0, e1));
        const double fl = kind == 0 ? 2.0 * 8 * iters * (double)nsm * thr : 2.0 * 8 * 8 * 4 * 4 * iters * (double)nsm * (thr / 32);
        if (rep) best = std::max(best, fl / (ms * 1e-3) * 1e-12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    *tflops = best;
    return RIS_OK;
}

extern "C" int ris_diag_gemm2_layout(ris_ctx* c, int32_t* ao_pos_host, int* panel_rows, int* tile_cols, int* ntiles, int* novf)
{
    if (!c) return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    if (ao_pos_host) {
        CU(cudaMemcpyAsync(ao_pos_host, c->d_ao_pos, sizeof(int) * (size_t)c->nao, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    if (panel_rows) *panel_rows = RIS_G2_BM;
    if (tile_cols) *tile_cols = RIS_G2_BN;
    if (ntiles) *ntiles = c->ntiles;
    if (novf) *novf = (int)std::min<long long>(c->g2_entries, 2147483647LL);
    return RIS_OK;
}

extern "C" int ris_probe_fp64_peak(double* tflops, void* cuda_stream) { return probe_fp64(0, tflops, cuda_stream); }
extern "C" int ris_probe_fp64_mma_peak(double* tflops, void* cuda_stream) { return probe_fp64(1, tflops, cuda_stream); }
