// ris_resp.cuh -- products of the ris coupling matrix with trial vectors (SURVEY.md 8(f) NEXT-3 and NEXT-4c): the
// excitation-energy stage (Casida / TDA, Eqs. 1-5 with the ris integrals of Eqs. 20-22) and the
// ris-approximated (A + B) of the Z-vector equation (Eq. 19; Sec. 4.2).  Included by ris_api.cu.
//
//   sigma[v]_ia = sum_jb [ cJ (ia|jb) - cKA (ij|ab) - cKB (ib|ja) ]^ris X[v]_jb,   (pq|sr)^ris = sum_AB (pq|A) M^-1_AB (B|sr)
//   A-coupling (Eq. 2): (1, c_x, 0);  B (Eq. 3): (1, 0, c_x);  A + B: (2, c_x, c_x);  A - B: (0, c_x, -c_x)
//
// ris_resp_setup stores, once per geometry and orbital set, the MO-basis three-index tensors ("reduced-size MO basis",
// PAPER.md:160) in the layouts the products read K-contiguously:
//   TJ  [f][i][a]          (ia|f) over the J-fit set (s and p functions)                 Coulomb term
//   Tvv [P][a][b']         (ab|P), rows padded to an even length                          (ij|ab): left factor of step 1
//   BooT[i][P][j']         sum_Q M^-1_PQ (ij|Q)                                           (ij|ab): left factor of step 2
//   Bov [P][i][b']         sum_Q M^-1_PQ (ib|Q)                                           (ib|ja): step 1
//   TovT[a][P][j']         (ja|P)                                                         (ib|ja): step 2
// and ris_resp_matvec evaluates, for a block of vectors,
//   Coulomb:   u[v][f] = sum_ia TJ[f][ia] X[v][ia];  w = M_J^-1 u (Cholesky);  sigma += cJ sum_f w[v][f] TJ[f][ia]
//              (two HBM-bound passes over TJ on the FP64 FMA pipes: 2 nvec flops per 8 bytes)
//   (ij|ab):   Y[v][a][P][j] = sum_b Tvv[P][a][b] X[v][j][b]          (DMMA GEMM, batched over P)
//              sigma[v][i][a] -= cKA sum_{P,j} BooT[i][P][j] Y[v][a][P][j]   (DMMA GEMM, K = naux*nocc split over P ranges)
//   (ib|ja):   Z[v][i][P][j] = sum_b Bov[P][i][b] X[v][j][b];  sigma[v][i][a] -= cKB sum_{P,j} Z[v][i][P][j] TovT[a][P][j]
// The split-K partial results are summed in a fixed order (deterministic).
#pragma once

// out[o0 ld0 + o1 ld1 + o2] (padding untouched) = in[o0 s0 + o1 s1 + o2 s2]
__global__ void ris_k_perm3(int n0, int n1, int n2, long long ld0, long long ld1, long long s0, long long s1, long long s2,
                            const double* __restrict__ in, double* __restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)n0 * n1 * n2) return;
    const int o2 = (int)(i % n2);
    const long long r = i / n2;
    const int o1 = (int)(r % n1), o0 = (int)(r / n1);
    out[o0 * ld0 + o1 * ld1 + o2] = in[o0 * s0 + o1 * s1 + o2 * s2];
}

// u partials: part[chunk][f][v] = sum_{k in chunk} TJ[f][k] X[v][k]  for FB functions x up to 8 vectors per block
constexpr int RIS_RESP_FB = 4, RIS_RESP_VB = 8;
__global__ void __launch_bounds__(256) ris_k_resp_ju(int nJ, long long nk, long long ldx, int nv8, long long kchunk,
                                                     const double* __restrict__ TJ, const double* __restrict__ X,
                                                     double* __restrict__ part)
{
    const int f0 = blockIdx.x * RIS_RESP_FB;
    const long long k0 = (long long)blockIdx.y * kchunk, k1 = min(nk, k0 + kchunk);
    double acc[RIS_RESP_FB][RIS_RESP_VB];
#pragma unroll
    for (int f = 0; f < RIS_RESP_FB; ++f)
#pragma unroll
        for (int v = 0; v < RIS_RESP_VB; ++v) acc[f][v] = 0.0;
    for (long long k = k0 + threadIdx.x; k < k1; k += blockDim.x) {
        double x[RIS_RESP_VB];
#pragma unroll
        for (int v = 0; v < RIS_RESP_VB; ++v) x[v] = v < nv8 ? X[v * ldx + k] : 0.0;
#pragma unroll
        for (int f = 0; f < RIS_RESP_FB; ++f) {
            const double t = f0 + f < nJ ? TJ[(size_t)(f0 + f) * nk + k] : 0.0;
#pragma unroll
            for (int v = 0; v < RIS_RESP_VB; ++v) acc[f][v] = fma(t, x[v], acc[f][v]);
        }
    }
    __shared__ double red[8][RIS_RESP_FB * RIS_RESP_VB];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int f = 0; f < RIS_RESP_FB; ++f)
#pragma unroll
        for (int v = 0; v < RIS_RESP_VB; ++v) {
            double a = acc[f][v];
            for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
            if (lane == 0) red[warp][f * RIS_RESP_VB + v] = a;
        }
    __syncthreads();
    if (threadIdx.x < RIS_RESP_FB * RIS_RESP_VB) {
        double a = 0.0;
        for (int w = 0; w < 8; ++w) a += red[w][threadIdx.x];
        const int f = threadIdx.x / RIS_RESP_VB, v = threadIdx.x % RIS_RESP_VB;
        if (f0 + f < nJ && v < nv8) part[((size_t)blockIdx.y * nJ + f0 + f) * RIS_RESP_VB + v] = a;
    }
}

// u[v][f] = sum_chunk part[chunk][f][v]   (fixed order)
__global__ void ris_k_resp_usum(int nJ, int nv8, int nchunk, const double* __restrict__ part, double* __restrict__ u)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nJ * nv8) return;
    const int v = i / nJ, f = i - v * nJ;
    double a = 0.0;
    for (int ch = 0; ch < nchunk; ++ch) a += part[((size_t)ch * nJ + f) * RIS_RESP_VB + v];
    u[(size_t)v * nJ + f] = a;
}

// sigma[v][k] = cJ sum_f w[v][f] TJ[f][k]   (overwrites; up to 8 vectors)
__global__ void __launch_bounds__(256) ris_k_resp_js(int nJ, long long nk, long long lds, int nv8, double cJ,
                                                     const double* __restrict__ TJ, const double* __restrict__ w,
                                                     double* __restrict__ sigma)
{
    constexpr int FT = 512;                 // functions per shared-memory tile of w
    __shared__ double sw[FT * RIS_RESP_VB];
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double acc[RIS_RESP_VB];
#pragma unroll
    for (int v = 0; v < RIS_RESP_VB; ++v) acc[v] = 0.0;
    for (int f0 = 0; f0 < nJ; f0 += FT) {
        const int nf = min(FT, nJ - f0);
        __syncthreads();
        for (int i = threadIdx.x; i < nf * RIS_RESP_VB; i += blockDim.x) {
            const int f = i / RIS_RESP_VB, v = i % RIS_RESP_VB;
            sw[i] = v < nv8 ? cJ * w[(size_t)v * nJ + f0 + f] : 0.0;
        }
        __syncthreads();
        if (k < nk)
            for (int f = 0; f < nf; ++f) {
                const double t = TJ[(size_t)(f0 + f) * nk + k];
#pragma unroll
                for (int v = 0; v < RIS_RESP_VB; ++v) acc[v] = fma(t, sw[f * RIS_RESP_VB + v], acc[v]);
            }
    }
    if (k >= nk) return;
#pragma unroll
    for (int v = 0; v < RIS_RESP_VB; ++v)
        if (v < nv8) sigma[v * lds + k] = acc[v];
}

// sigma[i] -= coef sum_z part[z][i]   (fixed order)
__global__ void ris_k_resp_sub_parts(long long n, int nz, double coef, const double* __restrict__ part, double* __restrict__ sigma)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double a = 0.0;
    for (int z = 0; z < nz; ++z) a += part[(size_t)z * n + i];
    sigma[i] = fma(-coef, a, sigma[i]);
}

extern "C" int ris_resp_free(ris_ctx* c)
{
    if (!c) return RIS_EINVAL;
    cudaStreamSynchronize(c->stream);
    RisResp& r = c->resp;
    for (double** p : {&r.TJ, &r.Tvv, &r.BooT, &r.Bov, &r.TovT, &r.Xp, &r.Y, &r.part, &r.uw})
        if (*p) { cudaFree(*p); *p = nullptr; }
    r = RisResp{};
    return RIS_OK;
}

static int resp_alloc(double** p, size_t n, bool zero, cudaStream_t st)
{
    cudaError_t e = cudaMalloc((void**)p, std::max<size_t>(n, 1) * sizeof(double));
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); *p = nullptr; return RIS_ENOMEM; }
    CU(e);
    if (zero) CU(cudaMemsetAsync(*p, 0, std::max<size_t>(n, 1) * sizeof(double), st));
    return RIS_OK;
}

extern "C" int ris_resp_setup(ris_ctx* c, int nocc, int nvir, const double* C_occ, const double* C_vir)
{
    if (!c || nocc < 1 || nvir < 1 || !C_occ || !C_vir) return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    ris_resp_free(c);
    RisResp& r = c->resp;
    const int nK = c->naux, nJ = c->naux_J;
    r.no = nocc; r.nv = nvir; r.nop = (nocc + 1) & ~1; r.nvp = (nvir + 1) & ~1;
    // split of the K = naux * nocc contraction over ranges of P: enough CTAs for one wave even with a single vector
    const int tiles1 = ((nocc + 63) / 64) * ((nvir + 127) / 128);
    r.nz = std::max(1, std::min(std::min(16, nK), (4 * c->nsm + tiles1 - 1) / tiles1));
    r.pc = (nK + r.nz - 1) / r.nz;
    r.nz = (nK + r.pc - 1) / r.pc;
    r.nKp = r.nz * r.pc;
    const size_t row = (size_t)r.nKp * r.nop;
    int rc;
    struct Guard { ris_ctx* c; bool ok = false; ~Guard() { if (!ok) ris_resp_free(c); } } guard{c};
    if ((rc = resp_alloc(&r.TJ, (size_t)nJ * nocc * nvir, false, c->stream))) return rc;
    if ((rc = resp_alloc(&r.Tvv, (size_t)nK * nvir * r.nvp, false, c->stream))) return rc;
    if ((rc = resp_alloc(&r.Bov, (size_t)nK * nocc * r.nvp, false, c->stream))) return rc;
    if ((rc = resp_alloc(&r.BooT, (size_t)nocc * row, true, c->stream))) return rc;
    if ((rc = resp_alloc(&r.TovT, (size_t)nvir * row, true, c->stream))) return rc;
    // Coulomb: (ia|f) over the J-fit set, no fit (the solve acts on u, naux_J numbers per vector)
    if ((rc = fit_mo(c, true, nocc, nvir, nvir, C_occ, C_vir, r.TJ, nullptr))) return rc;
    // exchange, s set: (ab|P) unfitted; (ib|P) fitted and unfitted; (ij|P) fitted
    if ((rc = fit_mo(c, false, nvir, nvir, r.nvp, C_vir, C_vir, r.Tvv, nullptr))) return rc;
    double *Tov, *Boo, *Too;
    if ((rc = ws_get(c, WS_RESP_T, sizeof(double) * (size_t)nK * nocc * std::max(r.nvp, r.nop), (void**)&Tov))) return rc;
    if ((rc = fit_mo(c, false, nocc, nvir, r.nvp, C_occ, C_vir, Tov, r.Bov))) return rc;
    const unsigned thr = 256;
    {   // TovT[a][P][j] = Tov[P][j][a]
        const long long n = (long long)nvir * nK * nocc;
        ris_k_perm3<<<(unsigned)((n + thr - 1) / thr), thr, 0, c->stream>>>(nvir, nK, nocc, (long long)row, r.nop, 1, (long long)nocc * r.nvp, r.nvp, Tov, r.TovT);
        CU(cudaGetLastError());
    }
    Too = Tov;
    if ((rc = ws_get(c, WS_RESP_B, sizeof(double) * (size_t)nK * nocc * r.nop, (void**)&Boo))) return rc;
    if ((rc = fit_mo(c, false, nocc, nocc, r.nop, C_occ, C_occ, Too, Boo))) return rc;
    {   // BooT[i][P][j] = Boo[P][i][j]
        const long long n = (long long)nocc * nK * nocc;
        ris_k_perm3<<<(unsigned)((n + thr - 1) / thr), thr, 0, c->stream>>>(nocc, nK, nocc, (long long)row, r.nop, r.nop, (long long)nocc * r.nop, 1, Boo, r.BooT);
        CU(cudaGetLastError());
    }
    if ((rc = metric_factor(c, true))) return rc;
    r.ready = true;
    guard.ok = true;
    return RIS_OK;
}

extern "C" int ris_resp_matvec(ris_ctx* c, int nvec, double cJ, double cKA, double cKB, const double* X, double* sigma)
{
    if (!c || nvec < 1 || !X || !sigma) return RIS_EINVAL;
    RisResp& r = c->resp;
    if (!r.ready) return RIS_EINVAL;
    CU(cudaSetDevice(c->device));
    const int nK = c->naux, nJ = c->naux_J, no = r.no, nv = r.nv, nop = r.nop, nvp = r.nvp;
    const long long nia = (long long)no * nv, row = (long long)r.nKp * nop, Kc = (long long)r.pc * nop;
    // vectors per pass: the Y / Z buffer (nv rows of naux*nocc per vector) within ~1/8 of the device memory
    size_t free_b = 0, total_b = 0;
    CU(cudaMemGetInfo(&free_b, &total_b));
    const size_t per_vec = sizeof(double) * (size_t)std::max(nv, no) * (size_t)row;
    int vc = (int)std::max<size_t>(1, std::min<size_t>((size_t)nvec, (total_b / 8) / per_vec));
    if (r.vc < vc || !r.Y) {
        CU(cudaStreamSynchronize(c->stream));
        for (double** p : {&r.Xp, &r.Y, &r.part, &r.uw})
            if (*p) { cudaFree(*p); *p = nullptr; }
        int rc;
        if ((rc = resp_alloc(&r.Xp, (size_t)vc * no * nvp, true, c->stream))) return rc;
        if ((rc = resp_alloc(&r.Y, (size_t)vc * std::max(nv, no) * (size_t)row, true, c->stream))) return rc;   // padding stays zero
        if ((rc = resp_alloc(&r.part, (size_t)r.nz * vc * nia, false, c->stream))) return rc;
        r.nchunk = (int)std::max<long long>(1, std::min<long long>(64, nia / 4096));
        if ((rc = resp_alloc(&r.uw, (size_t)(r.nchunk + 2) * nJ * RIS_RESP_VB, false, c->stream))) return rc;
        r.vc = vc;
    }
    vc = std::min(vc, r.vc);
    const unsigned thr = 256;
    for (int v0 = 0; v0 < nvec; v0 += vc) {
        const int nb = std::min(vc, nvec - v0);
        const double* Xs = X + (size_t)v0 * nia;
        double* sg = sigma + (size_t)v0 * nia;
        // ---- Coulomb term (also initialises sigma)
        if (cJ != 0.0) {
            double* part = r.uw;
            double* u = r.uw + (size_t)r.nchunk * nJ * RIS_RESP_VB;
            double* w = u + (size_t)nJ * RIS_RESP_VB;
            const long long kchunk = (nia + r.nchunk - 1) / r.nchunk;
            for (int b0 = 0; b0 < nb; b0 += RIS_RESP_VB) {
                const int n8 = std::min(RIS_RESP_VB, nb - b0);
                {
                    ProfScope ps(c, "ris_k_resp_ju", 2.0 * nJ * (double)nia * n8, 8.0 * (nJ + n8) * (double)nia);
                    ris_k_resp_ju<<<dim3((nJ + RIS_RESP_FB - 1) / RIS_RESP_FB, r.nchunk), 256, 0, c->stream>>>(
                        nJ, nia, nia, n8, kchunk, r.TJ, Xs + (size_t)b0 * nia, part);
                }
                ris_k_resp_usum<<<(nJ * n8 + 127) / 128, 128, 0, c->stream>>>(nJ, n8, r.nchunk, part, u);
                ris_k_chol_solve<<<n8, 256, sizeof(double) * nJ, c->stream>>>(nJ, c->jfit ? c->d_chol_J : c->d_chol, u, w);
                {
                    ProfScope ps(c, "ris_k_resp_js", 2.0 * nJ * (double)nia * n8, 8.0 * (nJ + n8) * (double)nia);
                    ris_k_resp_js<<<(unsigned)((nia + 255) / 256), 256, 0, c->stream>>>(
                        nJ, nia, nia, n8, cJ, r.TJ, w, sg + (size_t)b0 * nia);
                }
                CU(cudaGetLastError());
            }
        } else {
            CU(cudaMemsetAsync(sg, 0, sizeof(double) * (size_t)nb * nia, c->stream));
        }
        if (cKA == 0.0 && cKB == 0.0) continue;
        // X with even row length: Xp[(v,j)][nvp]
        {
            const long long n = (long long)nb * no * nvp;
            ris_k_pad2d<<<(unsigned)((n + thr - 1) / thr), thr, 0, c->stream>>>(nb * no, nv, nvp, Xs, r.Xp);
            CU(cudaGetLastError());
        }
        if (cKA != 0.0) {
            {   // Y[v][a][P][j] = sum_b Tvv[P][a][b] Xp[(v,j)][b]
                RisGemmParams g{};
                g.seg[0] = RisGemmSeg{r.Tvv, nvp, (long long)nv * nvp, r.Xp, nvp, 0, nv};
                g.nseg = 1; g.M = nv; g.N = nb * no; g.C = r.Y; g.ldc = row; g.bsC = nop;
                g.cdiv = no; g.cpad = (long long)nv * row;
                ProfScope ps(c, "ris_gemm_dmma(Y=Tvv*X^T)", 2.0 * nK * (double)nv * nv * no * nb, 8.0 * nK * ((double)nv * nv + (double)nv * no * nb));
                CU(ris_gemm_dense(c->stream, g, nK));
            }
            {   // part[z][v][i][a] = sum_{(P,j) in range z} BooT[i][(P,j)] Y[(v,a)][(P,j)]
                RisGemmParams g{};
                g.seg[0] = RisGemmSeg{r.BooT, row, Kc, r.Y, row, Kc, (int)Kc};
                g.nseg = 1; g.M = no; g.N = nb * nv; g.C = r.part; g.ldc = nv; g.bsC = (long long)nb * nia;
                g.cdiv = nv; g.cpad = nia;
                ProfScope ps(c, "ris_gemm_dmma(sigma-=Boo*Y^T)", 2.0 * nK * (double)no * no * nv * nb, 8.0 * ((double)no * row + (double)nv * row * nb));
                CU(ris_gemm_dense(c->stream, g, r.nz));
            }
            const long long n = (long long)nb * nia;
            ris_k_resp_sub_parts<<<(unsigned)((n + thr - 1) / thr), thr, 0, c->stream>>>(n, r.nz, cKA, r.part, sg);
            CU(cudaGetLastError());
        }
        if (cKB != 0.0) {
            {   // Z[v][i][P][j] = sum_b Bov[P][i][b] Xp[(v,j)][b]
                RisGemmParams g{};
                g.seg[0] = RisGemmSeg{r.Bov, nvp, (long long)no * nvp, r.Xp, nvp, 0, nv};
                g.nseg = 1; g.M = no; g.N = nb * no; g.C = r.Y; g.ldc = row; g.bsC = nop;
                g.cdiv = no; g.cpad = (long long)no * row;
                ProfScope ps(c, "ris_gemm_dmma(Z=Bov*X^T)", 2.0 * nK * (double)no * nv * no * nb, 8.0 * nK * ((double)no * nv + (double)no * no * nb));
                CU(ris_gemm_dense(c->stream, g, nK));
            }
            {   // part[z][v][i][a] = sum_{(P,j) in range z} Z[(v,i)][(P,j)] TovT[a][(P,j)]
                RisGemmParams g{};
                g.seg[0] = RisGemmSeg{r.Y, row, Kc, r.TovT, row, Kc, (int)Kc};
                g.nseg = 1; g.M = nb * no; g.N = nv; g.C = r.part; g.ldc = nv; g.bsC = (long long)nb * nia;
                ProfScope ps(c, "ris_gemm_dmma(sigma-=Z*Tov^T)", 2.0 * nK * (double)no * no * nv * nb, 8.0 * ((double)nv * row + (double)no * row * nb));
                CU(ris_gemm_dense(c->stream, g, r.nz));
            }
            const long long n = (long long)nb * nia;
            ris_k_resp_sub_parts<<<(unsigned)((n + thr - 1) / thr), thr, 0, c->stream>>>(n, r.nz, cKB, r.part, sg);
            CU(cudaGetLastError());
        }
    }
    return RIS_OK;
}
