/*
 * ris.h -- C ABI of the B200-native TDDFT-ris derivative-integral library (libris_b200.so).
 *
 * The library evaluates, on one NVIDIA B200 (sm_100a), the integral-derivative contractions of the
 * TDDFT-ris analytical excited-state gradient / derivative coupling (arxiv 2511.18233):
 *
 *   the derivative of the RI-factorised two-electron integral, Eq. 27,
 *       [sum_AB (pq|A) M^-1_AB (B|sr)]^xi = sum (pq|A)^xi M^-1 (B|sr) + sum (pq|A) M^-1 (B|sr)^xi
 *                                           - sum (pq|A) M^-1 M^xi M^-1 (B|sr),
 *   with the three-centre integrals (pq|A) and the metric M_AB = (A|B) of Eqs. 21-22
 *   over the minimal auxiliary basis (one GTO per angular-momentum component and atom; the paper's
 *   runs use s AND p functions for the Coulomb term and s functions only for exchange) -- the default set
 *   here is ONE s-type Gaussian per atom for both terms, ris_set_jfit gives the J-type calls an s + p set of their own --
 *   contracted with everything that is not an integral derivative:
 *
 *   ris_grad_J :  G[s][A][x] = sum_{mu nu} sum_P D^s_{mu nu} c^s_P  d(mu nu|P)/dR_{A,x}       (terms 1-2, Coulomb)
 *   ris_grad_K :  G[s][A][x] = sum_P sum_{mu nu} Gamma^{s,P}_{mu nu} d(mu nu|P)/dR_{A,x},
 *                 Gamma^{s,P} = C_occ B[s][P] C_vir^T   (terms 1-2, exchange; AO back-transform of
 *                 Eqs. 32-34, 39)
 *   ris_grad_PQ:  G[s][A][x] = sum_{PQ} c^s_P d^s_Q d(P|Q)/dR_{A,x}                          (term 3, POSITIVE sign)
 *
 * d/dR_A is the total nuclear derivative (xi is a nuclear coordinate, Eq. 8): every
 * centre sitting on atom A moves.  Physical prefactors (c_x of Eq. 21, closed-shell factors,
 * (E_J - E_I)^-1 of Eq. 26, the minus sign of term 3) are the caller's.
 *
 * Conventions
 *   - atomic units (bohr, Hartree/bohr); all arrays row-major, FP64 / int32; no hidden normalisation:
 *     prim_coef is applied as-is to UNnormalised Cartesian primitives
 *         phi(r) = sum_k d_k (x-A_x)^lx (y-A_y)^ly (z-A_z)^lz exp(-a_k |r-A|^2);
 *     the auxiliary function on atom P is N_P exp(-alpha_P |r-R_P|^2), N_P = (2 alpha_P/pi)^(3/4).
 *   - Cartesian component order inside a shell: lx descending, then ly descending
 *     (p: x,y,z; d: xx,xy,xz,yy,yz,zz; f: xxx,xxy,xxz,xyy,xyz,xzz,yyy,yyz,yzz,zzz).
 *     AO index = shells in input order, components in that order.
 *   - Pointers are HOST pointers in ris_setup and in the *_host entry points, DEVICE pointers (on the
 *     device current at ris_setup) in ris_grad_J / ris_grad_K / ris_grad_PQ.
 *   - Ownership: the caller owns every input and output buffer; the context owns its packed pair data
 *     and scratch and frees them in ris_destroy.  Outputs are OVERWRITTEN, not accumulated.
 *   - Asynchrony: device-pointer calls enqueue work on the stream given at ris_setup and return; the
 *     caller synchronises that stream.  *_host calls return after the result is in host memory.
 *     For small molecules (no angular-momentum class fills the GPU) a device-pointer call of ris_grad_J / ris_grad_K whose
 *     arguments repeat is captured into a CUDA graph on its second occurrence and replayed from then on: the same kernels in
 *     the same stream order, reading the buffers' current contents.
 *   - Errors: 0 on success, a negative ris_status otherwise; nothing aborts or throws across the ABI.
 *     There is no CPU fallback: without a usable CUDA device every call fails with RIS_ECUDA.
 */
#ifndef RIS_H
#define RIS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ris_ctx ris_ctx;

enum ris_status {
    RIS_OK = 0,
    RIS_EINVAL = -1,  /* bad argument: null pointer, l > 3, nprim < 1, index out of range, non-finite input */
    RIS_ENOMEM = -2,  /* host or device allocation failed */
    RIS_ECUDA = -3    /* CUDA runtime error; text via ris_strerror(RIS_ECUDA) */
};

typedef struct ris_options {
    double schwarz_tol;   /* screening threshold tau, default 1e-13; <= 0 disables screening.  tau bounds the
                             ACCUMULATED neglected contribution to a gradient component per unit |D c| / |Gamma|:
                             a primitive pair (a,b) of shell pair (mu,nu) is dropped when
                               |d_a d_b| K_ab (pi/p)^(3/2) max_P(N_P 2 pi/alpha_P) (1 + 2 max(a,b))
                                   < tau / (naux sqrt(n_unique_shell_pairs)),
                             (the bound on |(ab|P)| for s-type primitives -- the aux potential peaks at
                             N_P 2 pi/alpha_P -- times a factor for polynomial / derivative growth, with the
                             random-sign accumulation over naux x pairs folded into the threshold).  For l > 0 the
                             criterion is HEURISTIC: the polynomial prefactors |P-A|^la |P-B|^lb are not bounded
                             rigorously by the factor; it is validated empirically -- at tau = 1e-13 the results equal
                             the unscreened ones to 5e-15 of the gradient scale on configs 2-3 (tests/test_gpu_parity.py);
                             a shell pair is dropped when all its primitive pairs are.  There is no screening on
                             the aux index (the Coulomb tail is 1/R). */
    int deterministic;    /* nonzero: bitwise run-to-run reproducible results.  Every in-block sum already has a fixed
                             order; the cross-block sums then use 64-bit INTEGER atomics on a fixed-point split of
                             each contribution (value = hi 2^-28 + lo 2^-60; resolution 8.7e-19, contributions
                             |x| < 2^34, sums < 2^35 Hartree/bohr) instead of FP64 atomics.  A contribution outside
                             that range turns the whole output into NaN.  Default 0: FP64 atomics, run-to-run
                             differences at the 1e-16 relative level of the summation order. */
    int p_batch;          /* aux functions per Gamma^P batch in ris_grad_K; 0 = choose from free memory */
    int profile;          /* nonzero: record CUDA events around every kernel (see ris_profile_*) */
    int spherical;        /* nonzero: the caller's AO basis is spherical-harmonic (def2-TZVP):
                             shell s holds the 2l+1 functions S_lm(r - A) sum_k d_k exp(-a_k |r - A|^2), m = -l..l in this
                             order, S_lm = sqrt(4 pi/(2l+1)) r^l Y_lm^real the real regular solid harmonics in Racah
                             normalisation (S_1m = y, z, x; S_20 = zz - (xx + yy)/2; ...; the same prim_coef as the Cartesian
                             shell).  ris_nao() and every AO dimension of D, C_occ, C_vir then count sum (2l+1) functions; the
                             transformation to the Cartesian components the kernels run on happens on the device inside
                             each call.  Default 0: Cartesian shells. */
} ris_options;

/* Build the context: copies the molecule to the device and runs shell-pair screening, sorting by
 * (l_mu,l_nu) class and SoA packing ON THE DEVICE (north_star; the paper is silent).
 *   coords[natoms][3] bohr; shell s sits on atom shell_atom[s], has angular momentum shell_l[s] in 0..3 and
 *   1 <= shell_nprim[s] <= 24 primitives at prim_exp/prim_coef[shell_prim_off[s] ...] (RIS_EINVAL beyond); aux P sits on atom P with
 *   exponent aux_exponents[P] (bohr^-2).  opt may be NULL (defaults).  cuda_stream is a cudaStream_t
 *   (NULL = default stream) on which every later call of this context is enqueued. */
int ris_setup(ris_ctx** out, int natoms, const double* coords, int nshells, const int32_t* shell_atom,
              const int32_t* shell_l, const int32_t* shell_nprim, const int32_t* shell_prim_off,
              const double* prim_exp, const double* prim_coef, const double* aux_exponents,
              const ris_options* opt, void* cuda_stream);

/* J-type contraction.  D device [nbatch][nao][nao] (symmetric or not: only D + D^T contributes),
 * c_aux device [nbatch][naux_J] (naux_J = naux unless ris_set_jfit was called), grad device [nbatch][natoms][3]. */
int ris_grad_J(ris_ctx* ctx, int nbatch, const double* D, const double* c_aux, double* grad);

/* K-type contraction.  C_occ device [nao][nocc], C_vir device [nao][nvir] ("occ"/"vir" are just the
 * left / right coefficient matrices), B device [nbatch][naux][nocc][nvir], grad device [nbatch][natoms][3]. */
int ris_grad_K(ris_ctx* ctx, int nbatch, int nocc, int nvir, const double* C_occ, const double* C_vir,
               const double* B, double* grad);

/* Two-centre term.  c_aux, d_aux device [nbatch][naux_J], grad device [nbatch][natoms][3]. */
int ris_grad_PQ(ris_ctx* ctx, int nbatch, const double* c_aux, const double* d_aux, double* grad);

/* ---- Fitting step, J type (Eqs. 21-22) --------------------------------
 * ris_fit_J:   v[s][P] = sum_{mu nu} D^s_{mu nu} (mu nu|P)   (undifferentiated three-centre contraction, all ordered mu nu)
 *              c[s]    = M^-1 v[s],  M[P][Q] = N_P N_Q (P|Q)  (Cholesky factor built on the device by the first call,
 *                                                              kept in ctx)
 *   D device [nbatch][nao][nao] (any symmetry), v_out device [nbatch][naux] or NULL, c_out device [nbatch][naux].
 *   With these c, for fixed D:  d/dxi (1/2 v^T M^-1 v) = ris_grad_J(D, c) - 1/2 ris_grad_PQ(c, c)   (Eq. 27).
 *   RIS_EINVAL when the metric is not positive definite (coincident aux centres) or naux > 6144.
 * ris_metric:  M_out device [naux][naux], row-major, full (symmetric) matrix. */
int ris_fit_J(ris_ctx* ctx, int nbatch, const double* D, double* v_out, double* c_out);
int ris_metric(ris_ctx* ctx, double* M_out);

/* ---- Fitting step, K type (NEXT-1; Eqs. 21-22; MO-basis three-index tensor) ---------
 * ris_fit_K:  T[P][i][a] = sum_{mu nu} C_occ[mu,i] (mu nu|P) C_vir[nu,a]      (surviving shell pairs only)
 *             B[P][i][a] = sum_Q M^-1[P][Q] T[Q][i][a]                        -> the B that ris_grad_K takes (nbatch 1)
 *   C_occ device [nao][nocc], C_vir device [nao][nvir] (any two matrices with nao rows), T_out device
 *   [naux][nocc][nvir] or NULL, B_out device [naux][nocc][nvir].  Scratch (integral buffer, band slabs, half-transformed
 *   tensor: about 8 (naux nvir nao + naux * band) bytes) is ctx-owned.  For fixed C_occ, C_vir:
 *     d/dxi (1/2 sum_{PQ,ia} T^P_ia M^-1_PQ T^Q_ia) = ris_grad_K(C_occ, C_vir, B) - 1/2 ris_grad_PQ_full(G),
 *     G[P][Q] = sum_ia B[P][i][a] B[Q][i][a]                                  (Eq. 27).
 * ris_grad_PQ_full:  grad[s][A][x] = sum_{PQ} G[s][P][Q] d(P|Q)/dR_{A,x}  -- the metric term for a full matrix
 *   (SURVEY.md 8(c) A9); G device [nbatch][naux][naux] (any symmetry), grad device [nbatch][natoms][3], overwritten. */
int ris_fit_K(ris_ctx* ctx, int nocc, int nvir, const double* C_occ, const double* C_vir, double* T_out, double* B_out);
int ris_grad_PQ_full(ris_ctx* ctx, int nbatch, const double* G, double* grad);

/* The same three calls on HOST buffers: host->device copies, the kernels, and the device->host copy of
 * the gradient all happen inside the call, which returns when grad (host) is complete.  Pinned (page-locked) host
 * buffers let ris_grad_K_host stream B up in ranges of P on a second stream while the Gamma^P GEMMs of the
 * ranges already resident run; pageable buffers are accepted and simply copy synchronously. */
int ris_grad_J_host(ris_ctx* ctx, int nbatch, const double* D, const double* c_aux, double* grad);
int ris_grad_K_host(ris_ctx* ctx, int nbatch, int nocc, int nvir, const double* C_occ, const double* C_vir,
                    const double* B, double* grad);
int ris_grad_PQ_host(ris_ctx* ctx, int nbatch, const double* c_aux, const double* d_aux, double* grad);
/* All three terms in one call on host buffers (same argument meaning as above; nbatch_J states for D / c_aux / d_aux and
 * the J and PQ outputs, nbatch_K states for B and the K output).  The upload of B runs behind the J class kernels and the
 * GEMMs of the parts of B already resident; one synchronisation at the end. */
int ris_grad_host(ris_ctx* ctx, int nbatch_J, const double* D, const double* c_aux, const double* d_aux, int nbatch_K,
                  int nocc, int nvir, const double* C_occ, const double* C_vir, const double* B, double* grad_J,
                  double* grad_K, double* grad_PQ);

/* ---- Sharding over the auxiliary index (NEXT-4a) ------------------------------------------------------
 * Both three-centre contractions are sums over the auxiliary index, so the work of ONE state splits over GPUs by ranges of
 * it; the partial gradients add up to the full one (one all-reduce of nbatch natoms 3 doubles, done by the caller, e.g.
 * paper_2511_18233_b200/shard.py over NCCL).
 * ris_grad_K_range: the K-type contraction restricted to aux functions P in [p_lo, p_hi); B_local device
 *   [nbatch][p_hi - p_lo][nocc][nvir] holds ONLY this range (each GPU keeps its own slice of B); grad is overwritten with the
 *   partial result.  An empty range gives zeros.
 * ris_grad_J_range: the J-type contraction restricted to J-fit functions f in [f_lo, f_hi); c_aux keeps its full row
 *   length [nbatch][naux_J]. */
int ris_grad_K_range(ris_ctx* ctx, int nbatch, int nocc, int nvir, const double* C_occ, const double* C_vir,
                     const double* B_local, int p_lo, int p_hi, double* grad);
int ris_grad_J_range(ris_ctx* ctx, int nbatch, const double* D, const double* c_aux, int f_lo, int f_hi, double* grad);

/* ---- J-fit auxiliary set with p functions -----------------------------------
 * ris_set_jfit replaces, for the J-TYPE calls only (ris_grad_J, ris_fit_J, ris_grad_PQ and their *_host forms, ris_metric_J),
 * the default set by nshell_aux auxiliary SHELLS: shell k sits on atom aux_atom[k], has l = aux_l[k] in {0, 1} and exponent
 * aux_exp[k] (host arrays, copied).  The set's FUNCTIONS are the shells in input order, a p shell expanding into x, y, z:
 *     s:  N exp(-alpha |r-C|^2),            N = (2 alpha/pi)^(3/4)
 *     p:  N (r-C)_i exp(-alpha |r-C|^2),    N = (2 alpha/pi)^(3/4) 2 sqrt(alpha)      (unit self-overlap, as the s function)
 * c_aux / d_aux / v / c then have ris_naux_J() entries per state in that order.  The K-type calls (ris_grad_K, ris_fit_K,
 * ris_metric, ris_grad_PQ_full) keep the default s set, as in the paper's runs.  May be called again (new set);
 * RIS_EINVAL for l > 1, an atom out of range or a non-positive exponent.  ris_metric_J: M_out device [naux_J][naux_J]. */
int ris_set_jfit(ris_ctx* ctx, int nshell_aux, const int32_t* aux_atom, const int32_t* aux_l, const double* aux_exp);
int ris_naux_J(const ris_ctx* ctx);
int ris_metric_J(ris_ctx* ctx, double* M_out);

/* ---- Products of the ris coupling matrix with trial vectors (SURVEY.md 8(f) NEXT-3 and NEXT-4c) ------------------------
 * The excitation-energy stage (Casida / TDA: Eqs. 1-5 with the ris integrals of Eqs. 20-22; the
 * stored "reduced-size MO basis" tensors of PAPER.md:160) and the ris-approximated (A + B) of the Z-vector equation (Eq. 19,
 * PAPER.md:107; Sec. 4.2).  With i, j over the nocc columns of C_occ and a, b over the nvir columns of C_vir,
 *     sigma[v][i][a] = sum_jb [ cJ (ia|jb) - cKA (ij|ab) - cKB (ib|ja) ]^ris X[v][j][b],
 *     (pq|sr)^ris = sum_AB (pq|A) M^-1_AB (B|sr)   (Eq. 21; the Coulomb term over the J-fit set and its metric -- see
 *                                                   ris_set_jfit -- the two exchange terms over the default s set)
 *   coupling part of A (Eq. 2): (cJ, cKA, cKB) = (1, c_x, 0);  B (Eq. 3): (1, 0, c_x);  A + B: (2, c_x, c_x);  A - B: (0, c_x, -c_x).
 *   The orbital-energy diagonal of A and spin-adaptation factors (cJ = 2 for closed-shell singlets) are the caller's.
 * ris_resp_setup: C_occ device [nao][nocc], C_vir device [nao][nvir]; builds and keeps (ctx-owned, about
 *   8 (naux_J nocc nvir + naux (nvir^2 + 2 nocc nvir + nocc^2)) bytes) the MO-basis tensors (ia|f), (ab|P), M^-1 (ij|P),
 *   (ia|P), M^-1 (ia|P) in the layouts the products read; call it again after the orbitals change.  RIS_EINVAL when a metric
 *   is not positive definite or an auxiliary set has more than 6144 functions; RIS_ENOMEM when the tensors do not fit.
 * ris_resp_matvec: X, sigma device [nvec][nocc][nvir]; sigma is overwritten.  A zero coefficient skips its term.
 *   RIS_EINVAL before ris_resp_setup.  Deterministic (fixed summation order).
 * ris_resp_free releases the stored tensors (ris_destroy and ris_set_jfit do it too). */
int ris_resp_setup(ris_ctx* ctx, int nocc, int nvir, const double* C_occ, const double* C_vir);
int ris_resp_matvec(ris_ctx* ctx, int nvec, double cJ, double cKA, double cKB, const double* X, double* sigma);
int ris_resp_free(ris_ctx* ctx);

int ris_destroy(ris_ctx* ctx);
const char* ris_strerror(int status);

/* Queries (host values, valid after ris_setup). */
int ris_nao(const ris_ctx* ctx);
int ris_naux(const ris_ctx* ctx);
int ris_natoms(const ris_ctx* ctx);
long long ris_npairs(const ris_ctx* ctx, int la, int lb);      /* surviving unique shell pairs of class (la>=lb) */
long long ris_npairs_total(const ris_ctx* ctx);                /* unique shell pairs before screening */
long long ris_nprimpairs(const ris_ctx* ctx, int la, int lb);  /* surviving primitive pairs of the class */
long long ris_ntriplets(const ris_ctx* ctx);                   /* surviving primitive pairs x naux */
long long ris_ntriplets_unscreened(const ris_ctx* ctx);
long long ris_npair_elements(const ris_ctx* ctx);              /* packed Cartesian pair elements (no padding) */
int ris_p_batch(const ris_ctx* ctx);                           /* Gamma^P batch size chosen by the last ris_grad_K */

/* Profiling (opt.profile != 0): after synchronising the stream, ris_profile_count returns the number of
 * kernel launches recorded since the last ris_profile_reset; ris_profile_get returns launch i's kernel
 * name (static string) and device time in milliseconds. */
int ris_profile_reset(ris_ctx* ctx);
int ris_profile_enable(ris_ctx* ctx, int on);                   /* switch the recording on / off for the calls that follow */
int ris_profile_count(ris_ctx* ctx);
int ris_profile_get(ris_ctx* ctx, int i, const char** name, float* ms);
/* ALGORITHMIC work of launch i (what the method must compute / move, not what the kernel happens to do):
 * FP64 flops and HBM bytes, from the per-unit figures of DESIGN.md ("Algorithmic work per unit"). */
int ris_profile_get_work(ris_ctx* ctx, int i, double* flops, double* bytes);

#ifdef __cplusplus
}
#endif
#endif /* RIS_H */
