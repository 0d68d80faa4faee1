// nep_api.cu -- the C ABI of include/nep.h: host-side logic, allocation and kernel dispatch.
// Product code; never links, includes or calls anything under oracle/.
#include <math.h>
#include <stdlib.h>

#include <mutex>
#include <new>
#include <vector>

#include "nep_common.cuh"
#include "nep_neighbor.cuh"
#include "nep_kernels.cuh"
#include "nep_batch.cuh"
#include "nep_probe.cuh"

namespace {

const double kAccConv = 9.648533212e-3;   // (eV/Angstrom/amu) -> Angstrom/fs^2 (reading A10)
const double kBoltzmann = 8.617333262e-5; // eV/K (reading A10)

NepCoef make_coef()
{
    // Eqs. (13)-(16), (18), (19): closed forms of the pre-computed coefficients.
    NepCoef C;
    const double pi = 3.14159265358979323846;
    const double c3[NEP_NUM_S] = {
        3.0 / (4 * pi), 3.0 / (4 * pi), 3.0 / (4 * pi),
        5.0 / (16 * pi), 15.0 / (4 * pi), 15.0 / (4 * pi), 15.0 / (16 * pi), 15.0 / (16 * pi),
        7.0 / (16 * pi), 21.0 / (32 * pi), 21.0 / (32 * pi), 105.0 / (16 * pi), 105.0 / (16 * pi),
        35.0 / (32 * pi), 35.0 / (32 * pi),
        9.0 / (256 * pi), 45.0 / (32 * pi), 45.0 / (32 * pi), 45.0 / (64 * pi), 45.0 / (64 * pi),
        315.0 / (32 * pi), 315.0 / (32 * pi), 315.0 / (256 * pi), 315.0 / (256 * pi)};
    for (int k = 0; k < NEP_NUM_S; ++k) C.c3[k] = (float)c3[k];
    const double y20 = 0.25 * sqrt(5.0 / pi), y21 = 0.5 * sqrt(15.0 / (2 * pi)), y22 = 0.25 * sqrt(15.0 / (2 * pi));
    C.c4[0] = (float)(-sqrt(2.0 / 35.0) * y20 * y20 * y20);
    C.c4[1] = (float)(-6.0 * sqrt(1.0 / 70.0) * y20 * y21 * y21);
    C.c4[2] = (float)(6.0 * sqrt(2.0 / 35.0) * y20 * y22 * y22);
    C.c4[3] = (float)(6.0 * sqrt(3.0 / 35.0) * y21 * y21 * y22);
    C.c4[4] = (float)(-12.0 * sqrt(3.0 / 35.0) * y21 * y21 * y22);
    C.c5[0] = (float)(21.0 / (80 * pi * pi));
    C.c5[1] = (float)(21.0 / (40 * pi * pi));
    C.c5[2] = (float)(21.0 / (80 * pi * pi));
    return C;
}

int validate_hyper(const nep_hyper_t* h)
{
    if (!h) return NEP_ERR_INVALID_ARG;
    if (h->n_types < 1 || h->n_types > NEP_MAX_TYPES) return NEP_ERR_INVALID_ARG;
    if (!(h->rc_angular > 0.0) || !(h->rc_radial >= h->rc_angular)) return NEP_ERR_INVALID_ARG;
    if (h->n_max_radial < 0 || h->n_max_radial > 15 || h->n_max_angular < 0 || h->n_max_angular > 15) return NEP_ERR_INVALID_ARG;
    if (h->basis_radial < 0 || h->basis_radial > 31 || h->basis_angular < 0 || h->basis_angular > 31) return NEP_ERR_INVALID_ARG;
    if (h->l_max_3b != 4) return NEP_ERR_INVALID_ARG;
    if (h->l_max_4b != 0 && h->l_max_4b != 2) return NEP_ERR_INVALID_ARG;
    if (h->l_max_5b != 0 && h->l_max_5b != 1) return NEP_ERR_INVALID_ARG;
    if (h->n_neurons < 1 || h->n_neurons > 200) return NEP_ERR_INVALID_ARG;
    return NEP_OK;
}

int n_des(const nep_hyper_t* h)
{
    const int nblk = h->l_max_3b + (h->l_max_4b >= 2 ? 1 : 0) + (h->l_max_5b >= 1 ? 1 : 0);
    return (h->n_max_radial + 1) + (h->n_max_angular + 1) * nblk;     // Eq. (20)
}

void disown(nep_t* nep, void* p)
{
    for (int a = 0; a < nep->n_owned; ++a)
        if (nep->owned[a].p == p) { nep->owned[a] = nep->owned[--nep->n_owned]; return; }
}

template <typename T>
int dev_alloc(nep_t* nep, T** p, size_t count)
{
    if (*p) { disown(nep, *p); cudaFree(*p); *p = nullptr; }
    if (count == 0) count = 1;
    if (nep->n_owned >= (int)(sizeof(nep->owned) / sizeof(nep->owned[0]))) return nep_fail(nep, NEP_ERR_NOMEM, "allocation table full");
    cudaError_t e = cudaMalloc((void**)p, count * sizeof(T));
    if (e != cudaSuccess) {
        *p = nullptr;
        snprintf(nep->err, sizeof(nep->err), "cudaMalloc of %zu bytes failed: %s", count * sizeof(T), cudaGetErrorString(e));
        cudaGetLastError();
        return NEP_ERR_NOMEM;
    }
    nep->owned[nep->n_owned].p = *p;
    nep->owned[nep->n_owned].bytes = count * sizeof(T);
    nep->n_owned++;
    return NEP_OK;
}
#define NEP_TRY(x) do { int rc_ = (x); if (rc_ != NEP_OK) return rc_; } while (0)

// Shared memory is carved out of the 228 KB that also hold the L1 cache, and the driver sizes the
// carve-out for as many resident blocks as registers allow -- which can leave no L1 for the neighbour
// gathers.  cap_smem limits it to the blocks that fit in `budget` bytes (at least one).
template <typename K>
int cap_smem(nep_t* nep, K kernel, size_t bytes_per_block, size_t budget)
{
    const size_t per = bytes_per_block + 1024;            // + the driver's 1 KB per block
    size_t nb = budget / per;
    if (nb < 1) nb = 1;
    int pct = (int)((nb * per * 100 + 228 * 1024 - 1) / (228 * 1024));
    if (pct > 100) pct = 100;
    NEP_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, pct));
    return NEP_OK;
}

template <typename K>
int allow_smem(nep_t* nep, K kernel, size_t bytes)
{
    if (bytes > 48 * 1024) NEP_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return NEP_OK;
}

// ---- allocation ----------------------------------------------------------------------------------------
int alloc_lists(nep_t* nep, int capA, int capS)
{
    capA = (capA + 7) & ~7; capS = (capS + 7) & ~7;     // rows of the atom-major copy: whole 32-byte sectors
    if (capA > 256) capA = 256;
    if (capS > 256) capS = 256;
    const size_t n = (size_t)nep->n;
    nep->capA = nep->capS = nep->d.capA = nep->d.capS = 0;   // stay zero if an allocation below fails
    NEP_TRY(dev_alloc(nep, &nep->listA, (size_t)capA * n));
    NEP_TRY(dev_alloc(nep, &nep->rev, (size_t)capA * n));
    NEP_TRY(dev_alloc(nep, &nep->cA, (size_t)capA * n));
    NEP_TRY(dev_alloc(nep, &nep->pf, (size_t)capA * n));
    NEP_TRY(dev_alloc(nep, &nep->mA, (size_t)capA * n));
    NEP_TRY(dev_alloc(nep, &nep->listS, (size_t)capS * n));
    // the atom-major copy lives only during a build, when the per-step delivery buffers are free: it takes pf's storage
    // (16 capA n bytes) whenever 4 (capA + capS) n bytes fit there, which saves 0.35 GB at 1M atoms and 3.6 GB at 8.19M
    if ((size_t)(capA + capS) <= 4 * (size_t)capA) {
        if (nep->listT_own) { disown(nep, nep->listT_own); cudaFree(nep->listT_own); nep->listT_own = nullptr; }
        nep->listT = reinterpret_cast<int*>(nep->pf);
    } else {
        NEP_TRY(dev_alloc(nep, &nep->listT_own, (size_t)(capA + capS) * n));
        nep->listT = nep->listT_own;
    }
    NEP_TRY(dev_alloc(nep, &nep->revS, (size_t)capS * n));
    NEP_TRY(dev_alloc(nep, &nep->mB, (size_t)(capA + capS) * n));
    NEP_TRY(dev_alloc(nep, &nep->cB, (size_t)(capA + capS) * n));
    nep->capA = capA;
    nep->capS = capS;
    nep->d.capA = capA;
    nep->d.capS = capS;
    return NEP_OK;
}

int alloc_atoms(nep_t* nep, int64_t n)
{
    const size_t N = (size_t)n;
    const NepDims& d = nep->d;
    NEP_TRY(dev_alloc(nep, &nep->type_orig, N));
    NEP_TRY(dev_alloc(nep, &nep->perm, N));
    NEP_TRY(dev_alloc(nep, &nep->posq, N));
    NEP_TRY(dev_alloc(nep, &nep->posq_build, N));
    NEP_TRY(dev_alloc(nep, &nep->cell_of, N));
    NEP_TRY(dev_alloc(nep, &nep->rank_in_cell, N));
    NEP_TRY(dev_alloc(nep, &nep->cntA, N));
    NEP_TRY(dev_alloc(nep, &nep->cntS, N));
    NEP_TRY(dev_alloc(nep, &nep->ncA, N));
    NEP_TRY(dev_alloc(nep, &nep->ncB, N));
    NEP_TRY(dev_alloc(nep, &nep->fa, N));
    NEP_TRY(dev_alloc(nep, &nep->q, N * d.D));
    NEP_TRY(dev_alloc(nep, &nep->fp, N * d.D));
    NEP_TRY(dev_alloc(nep, &nep->S, N * d.NA * NEP_NUM_S));
    NEP_TRY(dev_alloc(nep, &nep->U, N));
    NEP_TRY(dev_alloc(nep, &nep->e_out, N));
    NEP_TRY(dev_alloc(nep, &nep->f_out, 3 * N));
    NEP_TRY(dev_alloc(nep, &nep->w_out, 9 * N));
    nep->atom_cap = n;
    nep->capA = nep->capS = 0;      // list storage is tied to n: force a re-allocation
    nep->mask_cap = 0;
    return NEP_OK;
}

// ---- neighbour build (used by nep_neighbors and by md_step rebuilds) -----------------------------------
int build_lists(nep_t* nep, const double* pos_dev)
{
    const int n = (int)nep->n;
    cudaStream_t st = nep->stream;
    const double rcut = nep->h.rc_radial + nep->skin, acut = nep->h.rc_angular + nep->skin;
    // the lists are overwritten from here on: nothing may use them (or an evaluation made with them) unless
    // this build succeeds
    nep->have_lists = nep->have_eval = nep->force_current = false;
    BuildParams P;
    P.n = n;
    P.n_types = nep->d.T;
    P.ncx = nep->ncell[0]; P.ncy = nep->ncell[1]; P.ncz = nep->ncell[2];
    P.ntx = nep->ntile[0]; P.nty = nep->ntile[1];
    P.hx = P.hy = P.hz = 2;
    CellInv inv;
    for (int a = 0; a < 9; ++a) { P.H[a] = nep->H[a]; P.Hinv[a] = nep->Hinv[a]; P.h[a] = nep->d.h[a]; inv.m[a] = nep->Hinv[a]; }
    P.tri = nep->d.tri;
    P.cutA2_d = acut * acut; P.cutR2_d = rcut * rcut;
    P.cutA2 = (float)P.cutA2_d; P.cutR2 = (float)P.cutR2_d;
    double Lmax = 0.0;                                   // |a| + |b| + |c| bounds every component's scale
    for (int k = 0; k < 3; ++k) Lmax += sqrt(P.H[3 * k] * P.H[3 * k] + P.H[3 * k + 1] * P.H[3 * k + 1] + P.H[3 * k + 2] * P.H[3 * k + 2]);
    // fp32/quantisation error of r^2 is < 2 r (3 L 2^-32 + r 2^-22); the band is ~100x wider
    P.guardR = (float)(1e-4 * P.cutR2_d + 64.0 * Lmax * rcut / 4294967296.0);
    P.guardA = (float)(1e-4 * P.cutA2_d + 64.0 * Lmax * acut / 4294967296.0);

    const int TB = 256;
    NEP_CUDA(cudaMemsetAsync(nep->cell_count, 0, sizeof(unsigned) * (size_t)(nep->n_cells + 1), st));
    NEP_LAUNCH(NEP_K_CELL_HIST, k_cell_hist<<<div_up(n, TB), TB, 0, st>>>(P, pos_dev, nep->cell_of, nep->rank_in_cell, nep->cell_count));
    {
        const int64_t m = nep->n_cells + 1;
        const int nb = div_up(m, SCAN_THREADS * SCAN_ITEMS);
        NEP_LAUNCH(NEP_K_SCAN, k_scan_blocks<<<nb, SCAN_THREADS, 0, st>>>(nep->cell_count, nep->cell_start, nep->scan_tmp, m));
        NEP_LAUNCH(NEP_K_SCAN, k_scan_totals<<<1, 1024, 0, st>>>(nep->scan_tmp, nb));
        NEP_LAUNCH(NEP_K_SCAN, k_scan_add<<<nb, SCAN_THREADS, 0, st>>>(nep->cell_start, nep->scan_tmp, m));
    }
    NEP_LAUNCH(NEP_K_SCATTER, k_scatter<<<div_up(n, TB), TB, 0, st>>>(n, nep->cell_of, nep->rank_in_cell, nep->cell_start, nep->perm));
    NEP_LAUNCH(NEP_K_SORT_CELLS, k_sort_cells<<<div_up(nep->n_cells, TB), TB, 0, st>>>(nep->n_cells, nep->cell_start, nep->perm));
    NEP_LAUNCH(NEP_K_QUANTIZE, k_quantize<<<div_up(n, TB), TB, 0, st>>>(n, pos_dev, nep->type_orig, nep->perm, inv, nep->posq));
    NEP_CUDA(cudaMemsetAsync(nep->disp_max, 0, 2 * sizeof(unsigned), st));

    if (nep->capA == 0) {   // first build for this n: size from the mean density, corrected below if short
        const double rho = (double)n / nep->volume;
        const double vA = 4.0 / 3.0 * 3.14159265358979 * acut * acut * acut, vR = 4.0 / 3.0 * 3.14159265358979 * rcut * rcut * rcut;
        // the outer shell gets the larger margin: its count per atom fluctuates more (a thin shell), and a re-allocation
        // in mid-run frees and allocates gigabytes with the device drained -- 20 ms to 1.2 s, measured
        int capA = (int)(rho * vA * 1.25) + 12, capS = (int)(rho * (vR - vA) * 1.6) + 16;
        if (capA > 256) capA = 256;
        NEP_TRY(alloc_lists(nep, capA, capS));
    }
    for (int attempt = 0; attempt < 4; ++attempt) {
        P.capA = nep->capA; P.capS = nep->capS;
        NEP_CUDA(cudaMemsetAsync(nep->flags, 0, sizeof(int) * 8, st));
        NEP_CUDA(cudaMemsetAsync(nep->build_stat, 0, sizeof(unsigned long long) * 2, st));
        if (P.tri) {
            NEP_LAUNCH(NEP_K_BUILD_LISTS, k_build_lists<true><<<div_up(n, 128), 128, 0, st>>>(P, pos_dev, nep->perm, nep->posq, nep->cell_start,
                                                              nep->listA, nep->cntA, nep->listS, nep->cntS, nep->flags, nep->build_stat));
        } else {
            NEP_LAUNCH(NEP_K_BUILD_LISTS, k_build_lists<false><<<div_up(n, 128), 128, 0, st>>>(P, pos_dev, nep->perm, nep->posq, nep->cell_start,
                                                               nep->listA, nep->cntA, nep->listS, nep->cntS, nep->flags, nep->build_stat));
        }
        int fl[8];
        unsigned long long stat[2];
        NEP_CUDA(cudaMemcpyAsync(fl, nep->flags, sizeof(fl), cudaMemcpyDeviceToHost, st));
        NEP_CUDA(cudaMemcpyAsync(stat, nep->build_stat, sizeof(stat), cudaMemcpyDeviceToHost, st));
        NEP_CUDA(cudaStreamSynchronize(st));
        nep->maxA_skin = fl[2];
        nep->maxR_skin = fl[3];
        nep->maxS_skin = fl[4];
        nep->raggedness = stat[1] > 0 ? (double)stat[0] / (double)stat[1] : 1.0;
        if (fl[5]) return nep_fail(nep, NEP_ERR_INVALID_ARG, "an atom type is outside [0, n_types)");
        if (fl[2] > (1 << NEP_SLOT_BITS)) return nep_fail(nep, NEP_ERR_NEIGHBOR_OVERFLOW, "more than 256 neighbours inside rc_angular + skin");
        if (fl[4] > (1 << NEP_SLOT_BITS)) return nep_fail(nep, NEP_ERR_NEIGHBOR_OVERFLOW, "more than 256 neighbours between rc_angular + skin and rc_radial + skin");
        if (!fl[0] && !fl[1]) break;
        if (attempt == 3) return nep_fail(nep, NEP_ERR_NEIGHBOR_OVERFLOW, "neighbour lists kept overflowing");
        // grow with a margin of a quarter: a re-allocation frees and allocates gigabytes and drains the device, so a
        // structure whose longest list keeps creeping up (a melt, a cluster) must not trigger one every few builds
        int capA = nep->capA, capS = nep->capS;
        if (fl[0]) capA = fl[2] + fl[2] / 4 + 8 > 256 ? 256 : fl[2] + fl[2] / 4 + 8;
        if (fl[1]) capS = fl[4] + fl[4] / 4 + 8 > 256 ? 256 : fl[4] + fl[4] / 4 + 8;
        NEP_TRY(alloc_lists(nep, capA, capS));
    }
    NEP_CUDA(cudaMemcpyAsync(nep->posq_build, nep->posq, sizeof(int4) * (size_t)n, cudaMemcpyDeviceToDevice, st));
    {
        const int row = nep->capA + nep->capS;
        NEP_LAUNCH(NEP_K_BUILD_REV, k_transpose_list<<<dim3(div_up(n, 32), div_up(nep->capA, 64)), 256, 0, st>>>(n, nep->capA, row, 0, nep->listA, nep->listT));
        NEP_LAUNCH(NEP_K_BUILD_REV, k_transpose_list<<<dim3(div_up(n, 32), div_up(nep->capS, 64)), 256, 0, st>>>(n, nep->capS, row, nep->capA, nep->listS, nep->listT));
    }
    NEP_LAUNCH(NEP_K_BUILD_REV, k_build_rev<<<div_up(n, 128), 128, 0, st>>>(n, nep->capA + nep->capS, 0, nep->listA, nep->cntA, nep->listT, nep->rev));
    NEP_LAUNCH(NEP_K_BUILD_REV, k_build_rev<<<div_up(n, 128), 128, 0, st>>>(n, nep->capA + nep->capS, nep->capA, nep->listS, nep->cntS, nep->listT, nep->revS));
    {
        const int longest = nep->maxA_skin > nep->maxS_skin ? nep->maxA_skin : nep->maxS_skin;
        nep->d.maskW = longest > 0 ? (longest + 63) / 64 : 1;
        nep->d.mrec = 4 * nep->d.maskW;
        if ((int64_t)n * nep->d.mrec > nep->mask_cap) {
            nep->mask_cap = 0;
            NEP_TRY(dev_alloc(nep, &nep->mask, (size_t)n * nep->d.mrec));
            nep->mask_cap = (int64_t)n * nep->d.mrec;
        }
    }
    nep->steps_since_build = 0;
    nep->have_lists = true;
    return NEP_OK;
}

// ---- one evaluation of (a2)-(a8) into the internal output buffers ---------------------------------------
const size_t kSmemTableMax = 96 * 1024;     // larger coefficient tables are read from global memory (L1)

// register variants (few species): TT * KP <= 64 and a coefficient table small enough to stage
const size_t kRegTableMax = 16 * 1024;

template <int TT, int KP>
int launch_radial_reg(nep_t* nep)
{
    const NepDims& d = nep->d;
    const size_t sm = sizeof(float) * (size_t)TT * TT * nep->strideR;
    NEP_LAUNCH(NEP_K_RADIAL, (k_radial_reg<TT, KP><<<div_up(d.n, 128), 128, sm, nep->stream>>>(d, nep->strideR, nep->posq, nep->cA, nep->ncA, nep->cB, nep->ncB,
                                                                              nep->cR_t, nep->q)));
    return NEP_OK;
}

template <int TT, int KP>
int launch_force_radial_reg(nep_t* nep)
{
    const NepDims& d = nep->d;
    const size_t sm = sizeof(float) * (size_t)TT * TT * d.NR * KP;
    NEP_LAUNCH(NEP_K_FORCE_RADIAL, (k_force_radial_reg<TT, KP><<<div_up(d.n, 128), 128, sm, nep->stream>>>(d, nep->posq, nep->cA, nep->ncA, nep->cB, nep->ncB, nep->mask,
                                                                                          nep->fp, nep->cR_e, nep->mA, nep->mB, nep->fa)));
    return NEP_OK;
}

// returns kNoVariant when (T, KP) has no register variant
const int kNoVariant = 1;
template <bool FORCE>
int dispatch_radial_reg(nep_t* nep)
{
    const NepDims& d = nep->d;
    if (d.T * nep->KP > 64 || d.T > 5) return kNoVariant;
    // the register variants spend T x KR select-FMAs per pair: beyond three species the shared-memory
    // variants (one row per pair) are faster (measured at T = 5: force 486 vs 523 us, descriptor 346 vs 355)
    if (d.T > 3) return kNoVariant;
    if (sizeof(float) * (size_t)d.T * d.T * nep->strideR > kRegTableMax) return kNoVariant;
    if (sizeof(float) * (size_t)d.T * d.T * d.NR * nep->KP > kRegTableMax) return kNoVariant;
#define NEP_REG_CASE(TT, KPV)                                                                      \
    if (d.T == TT && nep->KP == KPV) return FORCE ? launch_force_radial_reg<TT, KPV>(nep) : launch_radial_reg<TT, KPV>(nep);
    NEP_REG_CASE(1, 4) NEP_REG_CASE(1, 8) NEP_REG_CASE(1, 12) NEP_REG_CASE(1, 16) NEP_REG_CASE(1, 20) NEP_REG_CASE(1, 24) NEP_REG_CASE(1, 28) NEP_REG_CASE(1, 32)
    NEP_REG_CASE(2, 4) NEP_REG_CASE(2, 8) NEP_REG_CASE(2, 12) NEP_REG_CASE(2, 16) NEP_REG_CASE(2, 20) NEP_REG_CASE(2, 24) NEP_REG_CASE(2, 28) NEP_REG_CASE(2, 32)
    NEP_REG_CASE(3, 4) NEP_REG_CASE(3, 8) NEP_REG_CASE(3, 12) NEP_REG_CASE(3, 16) NEP_REG_CASE(3, 20)
    NEP_REG_CASE(4, 4) NEP_REG_CASE(4, 8) NEP_REG_CASE(4, 12) NEP_REG_CASE(4, 16)
    NEP_REG_CASE(5, 4) NEP_REG_CASE(5, 8) NEP_REG_CASE(5, 12)
#undef NEP_REG_CASE
    return kNoVariant;
}

// block size of the kernels that keep per-thread tables in shared memory: 128 threads, or 32 when the
// tables of 128 threads would not fit
const size_t kSmemBlockMax = 200 * 1024;

template <int KP, bool TAB_SM, int BS>
int launch_radial_multi2(nep_t* nep, size_t sm)
{
    const NepDims& d = nep->d;
    NEP_TRY(allow_smem(nep, k_radial_multi<KP, TAB_SM, BS>, sm));
    // one gather per pair and a read-modify-write of shared memory: occupancy matters more than L1 here
    NEP_TRY(cap_smem(nep, k_radial_multi<KP, TAB_SM, BS>, sm, (size_t)227 * 1024));
    NEP_LAUNCH(NEP_K_RADIAL, (k_radial_multi<KP, TAB_SM, BS><<<div_up(d.n, BS), BS, sm, nep->stream>>>(d, nep->strideR, nep->posq, nep->cA, nep->ncA,
                                                                                          nep->cB, nep->ncB, nep->cR_t, nep->q)));
    return NEP_OK;
}

template <int KP>
int launch_radial_multi(nep_t* nep)
{
    const NepDims& d = nep->d;
    const size_t tab_bytes = sizeof(float) * (size_t)d.T * d.T * nep->strideR;
    const bool tab_in_smem = tab_bytes <= kSmemTableMax;
    auto smem = [&](int b) { return sizeof(float) * (size_t)d.T * d.KR * b + (tab_in_smem ? tab_bytes : 0); };
    if (smem(128) <= kSmemBlockMax / 2)
        return tab_in_smem ? launch_radial_multi2<KP, true, 128>(nep, smem(128)) : launch_radial_multi2<KP, false, 128>(nep, smem(128));
    if (smem(32) > kSmemBlockMax) return nep_fail(nep, NEP_ERR_INVALID_ARG, "n_types x basis_radial too large for shared memory");
    return tab_in_smem ? launch_radial_multi2<KP, true, 32>(nep, smem(32)) : launch_radial_multi2<KP, false, 32>(nep, smem(32));
}

int dispatch_radial(nep_t* nep)
{
    if (!nep->force_smem_radial) { const int rc = dispatch_radial_reg<false>(nep); if (rc != kNoVariant) return rc; }
    switch (nep->KP) {
        case 4: return launch_radial_multi<4>(nep);
        case 8: return launch_radial_multi<8>(nep);
        case 12: return launch_radial_multi<12>(nep);
        case 16: return launch_radial_multi<16>(nep);
        case 20: return launch_radial_multi<20>(nep);
        case 24: return launch_radial_multi<24>(nep);
        case 28: return launch_radial_multi<28>(nep);
        case 32: return launch_radial_multi<32>(nep);
    }
    return nep_fail(nep, NEP_ERR_INVALID_ARG, "basis_radial out of range");
}

// resident blocks of a persistent (dynamic-tile) kernel: SMs x occupancy, at most one block per 128 atoms
template <typename K>
int persistent_grid(nep_t* nep, K kernel, size_t smem, int* grid)
{
    int per_sm = 0;
    NEP_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, 128, smem));
    if (per_sm < 1) per_sm = 1;
    *grid = (int)fmin((double)div_up(nep->d.n, 128), (double)per_sm * nep->num_sms);
    return NEP_OK;
}

template <int NCH, bool SM>
int launch_angular(nep_t* nep, const NepCoef& C, int p)
{
    const NepDims& d = nep->d;
    const int stride = nep->pass_stride[p], n0 = nep->pass_n0[p];
    const float* tab = nep->cA_t + nep->pass_off[p];
    const size_t sm = SM ? sizeof(float) * (size_t)d.T * d.T * stride : 0;
    int grid = 0;
    NEP_TRY(allow_smem(nep, k_angular<NCH, SM>, sm));
    NEP_TRY(persistent_grid(nep, k_angular<NCH, SM>, sm, &grid));
    NEP_LAUNCH(NEP_K_ANGULAR, (k_angular<NCH, SM><<<grid, 128, sm, nep->stream>>>(d, C, n0, stride, nep->posq, nep->cA, nep->ncA, tab, nep->S, nep->q,
                                                                                 nep->tile_ctr + p)));
    return NEP_OK;
}

// NCH channels with G in registers + NSM channels with G in shared memory (passes of 6 or 7 channels)
template <int NCH, int NSM, bool SM>
int launch_force_angular(nep_t* nep, const NepCoef& C, int p)
{
    const NepDims& d = nep->d;
    const int stride = nep->pass_stride[p], n0 = nep->pass_n0[p];
    const float* tab = nep->cA_t + nep->pass_off[p];
    const size_t sm = (SM ? sizeof(float) * (size_t)d.T * d.T * stride : 0) + sizeof(float) * (size_t)NSM * NEP_NUM_S * 128;
    int grid = 0;
    NEP_TRY(allow_smem(nep, k_force_angular<NCH, NSM, SM>, sm));
    NEP_TRY(persistent_grid(nep, k_force_angular<NCH, NSM, SM>, sm, &grid));
    NEP_LAUNCH(NEP_K_FORCE_ANGULAR, (k_force_angular<NCH, NSM, SM><<<grid, 128, sm, nep->stream>>>(d, C, n0, p > 0, stride, nep->posq, nep->cA, nep->ncA, nep->mask, tab,
                                                                                                  nep->S, nep->fp, nep->pf, nep->fa, nep->tile_ctr + 16 + p)));
    return NEP_OK;
}

int dispatch_angular(nep_t* nep, const NepCoef& C, bool force_pass)
{
    for (int p = 0; p < nep->n_pass; ++p) {
        int rc;
        if (!nep->angular_tab_smem) rc = force_pass ? launch_force_angular<4, 0, false>(nep, C, p) : launch_angular<4, false>(nep, C, p);
        else if (!force_pass) switch (nep->pass_nch[p]) {
            case 1: rc = launch_angular<1, true>(nep, C, p); break;
            case 2: rc = launch_angular<2, true>(nep, C, p); break;
            case 3: rc = launch_angular<3, true>(nep, C, p); break;
            case 4: rc = launch_angular<4, true>(nep, C, p); break;
            case 5: rc = launch_angular<5, true>(nep, C, p); break;
            case 6: rc = launch_angular<6, true>(nep, C, p); break;
            default: rc = launch_angular<7, true>(nep, C, p); break;
        }
        else switch (nep->pass_nch[p]) {
            case 1: rc = launch_force_angular<1, 0, true>(nep, C, p); break;
            case 2: rc = launch_force_angular<2, 0, true>(nep, C, p); break;
            case 3: rc = launch_force_angular<3, 0, true>(nep, C, p); break;
            case 4: rc = launch_force_angular<4, 0, true>(nep, C, p); break;
            case 5: rc = launch_force_angular<5, 0, true>(nep, C, p); break;
            case 6: rc = launch_force_angular<5, 1, true>(nep, C, p); break;
            default: rc = launch_force_angular<5, 2, true>(nep, C, p); break;
        }
        if (rc != NEP_OK) return rc;
    }
    return NEP_OK;
}

template <int DP>
int launch_ann(nep_t* nep)
{
    const NepDims& d = nep->d;
    int bs = 128;                                        // smaller blocks for networks whose weights fill shared memory
    auto smem = [&](int b) { return sizeof(float) * ((size_t)d.H * DP + 2 * d.H + (size_t)d.H * b); };
    while (bs > 32 && smem(bs) > 110 * 1024) bs >>= 1;
    const size_t sm = smem(bs);
    NEP_TRY(allow_smem(nep, k_ann<DP>, sm));
    NEP_LAUNCH(NEP_K_ANN, k_ann<DP><<<div_up(d.n, bs), bs, sm, nep->stream>>>(d, nep->q, nep->w0p, nep->b0, nep->w1, nep->b1, nep->fp, nep->U));
    return NEP_OK;
}

// tensor-core variant (3xTF32): descriptor tiers up to 72, weights + per-warp tiles within 100 KB of shared memory
template <int DP>
int launch_ann_tc(nep_t* nep, bool* done)
{
    const NepDims& d = nep->d;
    const int HP = (d.H + 7) & ~7;
    const size_t sm = sizeof(float) * ((size_t)2 * HP * ann_stride_fwd(DP) + (size_t)2 * HP * ann_stride_bwd(DP) + 2 * HP + (size_t)4 * 32 * (HP + 4));
    *done = false;
    if (sm > 100 * 1024) return NEP_OK;
    NEP_TRY(allow_smem(nep, k_ann_tc<DP>, sm));
    int grid = 0;
    NEP_TRY(persistent_grid(nep, k_ann_tc<DP>, sm, &grid));
    NEP_LAUNCH(NEP_K_ANN, k_ann_tc<DP><<<grid, 128, sm, nep->stream>>>(d, HP, nep->q, nep->w0p, nep->b0, nep->w1, nep->b1, nep->fp, nep->U, nep->tile_ctr + 32));
    *done = true;
    return NEP_OK;
}

int ann_tier(int D)
{
    const int tiers[] = {24, 40, 56, 72, 88, 104, 120};
    for (int t : tiers) if (D <= t) return t;
    return -1;
}

int dispatch_ann(nep_t* nep)
{
    if (!nep->ann_fp32 && !nep->ann_precise) {
        bool done = false;
        int rc = NEP_OK;
        switch (nep->DP) {
            case 24: rc = launch_ann_tc<24>(nep, &done); break;
            case 40: rc = launch_ann_tc<40>(nep, &done); break;
            case 56: rc = launch_ann_tc<56>(nep, &done); break;
            case 72: rc = launch_ann_tc<72>(nep, &done); break;
        }
        if (rc != NEP_OK || done) return rc;
    }
    switch (nep->DP) {
        case 24: return launch_ann<24>(nep);
        case 40: return launch_ann<40>(nep);
        case 56: return launch_ann<56>(nep);
        case 72: return launch_ann<72>(nep);
        case 88: return launch_ann<88>(nep);
        case 104: return launch_ann<104>(nep);
        case 120: return launch_ann<120>(nep);
    }
    return nep_fail(nep, NEP_ERR_INVALID_ARG, "descriptor too long");
}

template <int KP, bool TAB_SM, int BS>
int launch_force_radial2(nep_t* nep, size_t sm)
{
    const NepDims& d = nep->d;
    NEP_TRY(allow_smem(nep, k_force_radial<KP, TAB_SM, BS>, sm));
    NEP_TRY(cap_smem(nep, k_force_radial<KP, TAB_SM, BS>, sm, nep->smem_budget));
    NEP_LAUNCH(NEP_K_FORCE_RADIAL, (k_force_radial<KP, TAB_SM, BS><<<div_up(d.n, BS), BS, sm, nep->stream>>>(d, nep->posq, nep->cA, nep->ncA, nep->cB, nep->ncB, nep->mask,
                                                                                                nep->fp, nep->cR_e, nep->mA, nep->mB, nep->fa)));
    return NEP_OK;
}

template <int KP>
int launch_force_radial(nep_t* nep)
{
    const NepDims& d = nep->d;
    const size_t tab_bytes = sizeof(float) * (size_t)d.T * d.T * d.NR * KP;
    const bool tab_in_smem = tab_bytes <= kSmemTableMax;
    auto smem = [&](int b) { return sizeof(float) * (size_t)round_up4(d.T * d.KR) * b + (tab_in_smem ? tab_bytes : 0); };
    if (smem(128) <= kSmemBlockMax / 2)
        return tab_in_smem ? launch_force_radial2<KP, true, 128>(nep, smem(128)) : launch_force_radial2<KP, false, 128>(nep, smem(128));
    if (smem(32) > kSmemBlockMax) return nep_fail(nep, NEP_ERR_INVALID_ARG, "n_types x basis_radial too large for shared memory");
    return tab_in_smem ? launch_force_radial2<KP, true, 32>(nep, smem(32)) : launch_force_radial2<KP, false, 32>(nep, smem(32));
}

int dispatch_force_radial(nep_t* nep)
{
    if (!nep->force_smem_radial) { const int rc = dispatch_radial_reg<true>(nep); if (rc != kNoVariant) return rc; }
    switch (nep->KP) {
        case 4: return launch_force_radial<4>(nep);
        case 8: return launch_force_radial<8>(nep);
        case 12: return launch_force_radial<12>(nep);
        case 16: return launch_force_radial<16>(nep);
        case 20: return launch_force_radial<20>(nep);
        case 24: return launch_force_radial<24>(nep);
        case 28: return launch_force_radial<28>(nep);
        case 32: return launch_force_radial<32>(nep);
    }
    return nep_fail(nep, NEP_ERR_INVALID_ARG, "basis_radial out of range");
}

int dispatch_final(nep_t* nep)
{
    const NepDims& d = nep->d;
    NEP_LAUNCH(NEP_K_FINAL, k_final<<<div_up(d.n, 256), 256, 0, nep->stream>>>(d, nep->posq, nep->perm, nep->cA, nep->ncA, nep->cB, nep->ncB, nep->pf, nep->mA, nep->mB,
                                                       nep->fa, nep->U, nep->e_out, nep->f_out, nep->w_out));
    return NEP_OK;
}

int evaluate(nep_t* nep, const double* pos_dev, bool reuse_geometry = false)
{
    static const NepCoef C = make_coef();
    const NepDims& d = nep->d;
    const int n = d.n;
    cudaStream_t st = nep->stream;
    CellInv inv;
    for (int a = 0; a < 9; ++a) inv.m[a] = nep->Hinv[a];
    NEP_CUDA(cudaMemsetAsync(nep->tile_ctr, 0, sizeof(int) * 64, st));
    if (!reuse_geometry) {   // else: same positions as the previous evaluation (another member of a population)
        NEP_LAUNCH(NEP_K_QUANTIZE, k_quantize<<<div_up(n, 256), 256, 0, st>>>(n, pos_dev, nep->type_orig, nep->perm, inv, nep->posq));
        NEP_CUDA(cudaMemsetAsync(nep->disp_max, 0, sizeof(unsigned), st));   // [0] only: [1] runs since the build
        if (n <= (1 << 22)) {
            NEP_LAUNCH(NEP_K_FILTER, k_filter<true><<<div_up(n, 256), 256, 0, st>>>(d, nep->posq, nep->posq_build, nep->listA, nep->cntA, nep->rev, nep->listS, nep->cntS,
                                                           nep->revS, nep->cA, nep->ncA, nep->cB, nep->ncB, nep->mask, nep->disp_max));
        } else {
            NEP_LAUNCH(NEP_K_FILTER, k_filter<false><<<div_up(n, 256), 256, 0, st>>>(d, nep->posq, nep->posq_build, nep->listA, nep->cntA, nep->rev, nep->listS, nep->cntS,
                                                            nep->revS, nep->cA, nep->ncA, nep->cB, nep->ncB, nep->mask, nep->disp_max));
        }
    }
    NEP_TRY(dispatch_radial(nep));
    NEP_TRY(dispatch_angular(nep, C, false));
    NEP_TRY(dispatch_ann(nep));
    NEP_TRY(dispatch_angular(nep, C, true));
    NEP_TRY(dispatch_force_radial(nep));
    NEP_TRY(dispatch_final(nep));
    nep->have_eval = true;
    return NEP_OK;
}

int setup_system(nep_t* nep, int64_t n, const double box[9], double skin)
{
    if (n <= 0 || n > NEP_MAX_ATOMS || !box || !(skin >= 0.0)) return nep_fail(nep, NEP_ERR_INVALID_ARG, "bad n, box or skin");
    // cell rows a, b, c; inverse by cofactors; perpendicular widths w_k = 1 / |column k of Hinv|
    const double* H = box;
    for (int a = 0; a < 9; ++a)
        if (!(H[a] == H[a]) || fabs(H[a]) > 1e12) return nep_fail(nep, NEP_ERR_INVALID_ARG, "bad box");
    const double c00 = H[4] * H[8] - H[5] * H[7], c01 = H[5] * H[6] - H[3] * H[8], c02 = H[3] * H[7] - H[4] * H[6];
    const double det = (H[0] * c00 + H[1] * c01) + H[2] * c02;
    if (!(det > 0.0)) return nep_fail(nep, NEP_ERR_UNSUPPORTED_BOX, "the cell vectors a, b, c must form a right-handed, non-degenerate cell");
    double inv[9];
    inv[0] = c00 / det; inv[1] = (H[2] * H[7] - H[1] * H[8]) / det; inv[2] = (H[1] * H[5] - H[2] * H[4]) / det;
    inv[3] = c01 / det; inv[4] = (H[0] * H[8] - H[2] * H[6]) / det; inv[5] = (H[2] * H[3] - H[0] * H[5]) / det;
    inv[6] = c02 / det; inv[7] = (H[1] * H[6] - H[0] * H[7]) / det; inv[8] = (H[0] * H[4] - H[1] * H[3]) / det;
    double width[3];
    for (int k = 0; k < 3; ++k) width[k] = 1.0 / sqrt(inv[k] * inv[k] + inv[3 + k] * inv[3 + k] + inv[6 + k] * inv[6 + k]);
    const double rcut = nep->h.rc_radial + skin;
    for (int k = 0; k < 3; ++k)
        if (!(width[k] >= 2.0 * rcut)) return nep_fail(nep, NEP_ERR_BOX_TOO_SMALL, "a perpendicular width of the cell < 2 (rc_radial + skin)");
    const bool same_n = (n == nep->n);
    nep->skin = skin;
    nep->volume = det;
    nep->d.tri = 0;
    for (int a = 0; a < 9; ++a) {
        nep->H[a] = H[a];
        nep->Hinv[a] = inv[a];
        nep->d.h[a] = (float)(H[a] / 4294967296.0);
        if (a % 4 != 0 && H[a] != 0.0) nep->d.tri = 1;
    }
    int64_t nc = 1;
    const double cell_min = 0.5 * rcut * (1.0 + 1e-6);
    for (int a = 0; a < 3; ++a) {                       // cells are slabs in fractional space: thickness width / nc
        int c = (int)floor(width[a] / cell_min);
        if (c < 1) c = 1;
        if (c > 1024) c = 1024;
        nep->ncell[a] = c;
        nep->ntile[a] = (c + 3) / 4;
        nc *= 4 * (int64_t)nep->ntile[a];
    }
    nep->n_cells = nc;
    nep->raggedness = 1.0;
    if (!same_n || n > nep->atom_cap) {
        nep->n = n;
        nep->d.n = (int)n;
        NEP_TRY(alloc_atoms(nep, n));
    }
    if (nc + 1 > nep->cell_cap) {
        NEP_TRY(dev_alloc(nep, &nep->cell_count, (size_t)nc + 1));
        NEP_TRY(dev_alloc(nep, &nep->cell_start, (size_t)nc + 1));
        nep->cell_cap = nc + 1;
    }
    const int64_t nb = div_up(nc + 1, SCAN_THREADS * SCAN_ITEMS);
    if (nb > nep->scan_cap) {
        NEP_TRY(dev_alloc(nep, &nep->scan_tmp, (size_t)nb));
        nep->scan_cap = nb;
    }
    return NEP_OK;
}

template <int DP>
int launch_batch_ann2(nep_t* nep, dim3 grid, const BatchParams& P, double* energy_dev)
{
    const NepDims& d = nep->d;
    const size_t sm = sizeof(float) * ((size_t)d.H * DP + 2 * d.H + (size_t)d.H * 128);
    NEP_TRY(allow_smem(nep, kb_ann<DP>, sm));
    NEP_LAUNCH(NEP_K_BATCH_ANN, kb_ann<DP><<<grid, 128, sm, nep->stream>>>(d, nep->b.N, P, nep->b.q, nep->b.fp, energy_dev));
    return NEP_OK;
}

int launch_batch_ann(nep_t* nep, dim3 grid, const BatchParams& P, double* energy_dev)
{
    switch (nep->DP) {
        case 24: return launch_batch_ann2<24>(nep, grid, P, energy_dev);
        case 40: return launch_batch_ann2<40>(nep, grid, P, energy_dev);
        case 56: return launch_batch_ann2<56>(nep, grid, P, energy_dev);
        case 72: return launch_batch_ann2<72>(nep, grid, P, energy_dev);
        case 88: return launch_batch_ann2<88>(nep, grid, P, energy_dev);
        case 104: return launch_batch_ann2<104>(nep, grid, P, energy_dev);
        case 120: return launch_batch_ann2<120>(nep, grid, P, energy_dev);
    }
    return nep_fail(nep, NEP_ERR_INVALID_ARG, "descriptor too long");
}

template <int DP>
int launch_latent(nep_t* nep, float* latent_dev)
{
    const NepDims& d = nep->d;
    const size_t sm = sizeof(float) * ((size_t)d.H * DP + 2 * d.H);
    NEP_TRY(allow_smem(nep, k_latent<DP>, sm));
    NEP_LAUNCH(NEP_K_EXPORT, k_latent<DP><<<div_up(d.n, 128), 128, sm, nep->stream>>>(d, nep->perm, nep->q, nep->w0p, nep->b0, nep->w1, latent_dev));
    return NEP_OK;
}

// Re-laid-out parameter tables (layouts documented at the kernels that read them) from the caller's host
// arrays; device arrays are allocated on first use.  Copies are enqueued on the handle's stream and the
// stream is synchronised (the host vectors are temporaries), so a later evaluation sees the new model.
int upload_parameters(nep_t* nep, const float* c_radial, const float* c_angular, const float* w0, const float* b0,
                      const float* w1, const float* b1)
{
    const NepDims& d = nep->d;
    const int TT = d.T * d.T;
    std::vector<float> cRt((size_t)TT * nep->strideR, 0.0f);
    std::vector<float> cAt((size_t)nep->pass_off[nep->n_pass - 1] + (size_t)TT * nep->pass_stride[nep->n_pass - 1], 0.0f);
    std::vector<float> cRe((size_t)TT * d.NR * d.KRP, 0.0f), w0p((size_t)d.H * nep->DP, 0.0f);
    for (int tt = 0; tt < TT; ++tt) {
        for (int nn = 0; nn < d.NR; ++nn)
            for (int k = 0; k < d.KR; ++k) {
                const float v = c_radial[((size_t)tt * d.NR + nn) * d.KR + k];
                cRt[(size_t)tt * nep->strideR + (size_t)k * d.NRP + nn] = v;
                cRe[((size_t)tt * d.NR + nn) * d.KRP + k] = v;
            }
        for (int p = 0; p < nep->n_pass; ++p) {
            const int NCHP = round_up4(nep->pass_nch[p]);
            float* tab = cAt.data() + nep->pass_off[p] + (size_t)tt * nep->pass_stride[p];
            for (int a = 0; a < nep->pass_nch[p] && nep->pass_n0[p] + a < d.NA; ++a) {
                const float* c = c_angular + ((size_t)tt * d.NA + nep->pass_n0[p] + a) * d.KA;
                double csum = 2.0 * (double)c[0];                  // csum'_n = 2 c_n0 + sum_{k>=1} c_nk
                for (int k = 1; k < d.KA; ++k) {
                    tab[(size_t)k * NCHP + a] = c[k];
                    csum += (double)c[k];
                }
                tab[a] = (float)csum;
            }
        }
    }
    for (int m = 0; m < d.H; ++m)
        for (int v = 0; v < d.D; ++v) w0p[(size_t)m * nep->DP + v] = w0[(size_t)m * d.D + v];
    nep->b1 = b1[0];
    std::vector<float> vb0(b0, b0 + d.H), vw1(w1, w1 + d.H);
    // k_ann_tc evaluates tanh with MUFU.EX2 / MUFU.RCP (tanh_fast: absolute error ~1e-7 per neuron), so its error in
    // U_i is bounded by sum_m |w1_m| x 1e-7.  Up to sum |w1| = 5 that is 5e-7 eV, a twentieth of north_star's 1e-5 eV
    // bar; wider or larger-weight output layers (trained |w1| > 1, up to 200 neurons) take the tanhf kernel instead.
    double w1_abs = 0.0;
    for (int m = 0; m < d.H; ++m) w1_abs += fabs((double)w1[m]);
    nep->ann_precise = w1_abs > 5.0;
#define UPLOAD(dst, vec)                                                                          \
    do {                                                                                          \
        if (!nep->dst) NEP_TRY(dev_alloc(nep, &nep->dst, (vec).size()));                          \
        NEP_CUDA(cudaMemcpyAsync(nep->dst, (vec).data(), (vec).size() * sizeof((vec)[0]), cudaMemcpyHostToDevice, nep->stream)); \
    } while (0)
    UPLOAD(cR_t, cRt);
    UPLOAD(cA_t, cAt);
    UPLOAD(cR_e, cRe);
    UPLOAD(w0p, w0p);
    UPLOAD(b0, vb0);
    UPLOAD(w1, vw1);
#undef UPLOAD
    NEP_CUDA(cudaStreamSynchronize(nep->stream));
    return NEP_OK;
}

}  // namespace

// =======================================================================================================
extern "C" {

const char* nep_status_string(int status)
{
    switch (status) {
        case NEP_OK: return "ok";
        case NEP_ERR_INVALID_ARG: return "invalid argument";
        case NEP_ERR_BOX_TOO_SMALL: return "box too small for the cutoff (minimum image)";
        case NEP_ERR_UNSUPPORTED_BOX: return "unsupported box (degenerate or left-handed cell)";
        case NEP_ERR_NEIGHBOR_OVERFLOW: return "neighbour list overflow";
        case NEP_ERR_STATE: return "call out of order";
        case NEP_ERR_CUDA: return "CUDA error";
        case NEP_ERR_NOMEM: return "out of memory";
        case NEP_ERR_SKIN_EXCEEDED: return "an atom moved more than skin/2 between two list builds";
    }
    return "unknown status";
}

const char* nep_last_error(const nep_t* nep) { return nep ? nep->err : "null handle"; }

int64_t nep_launch_count(const nep_t* nep) { return nep ? nep->launches : 0; }

int nep_num_descriptors(const nep_hyper_t* h)
{
    const int rc = validate_hyper(h);
    return rc != NEP_OK ? rc : n_des(h);
}

int nep_create(nep_t** out, const nep_hyper_t* h, const float* c_radial, const float* c_angular,
               const float* w0, const float* b0, const float* w1, const float* b1,
               const double* mass_amu, int device, void* cuda_stream)
{
    if (!out) return NEP_ERR_INVALID_ARG;
    *out = nullptr;
    int rc = validate_hyper(h);
    if (rc != NEP_OK) return rc;
    if (!c_radial || !c_angular || !w0 || !b0 || !w1 || !b1 || !mass_amu) return NEP_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return NEP_ERR_CUDA; }
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return NEP_ERR_CUDA; }

    nep_t* nep = new (std::nothrow) nep_ctx();
    if (!nep) return NEP_ERR_NOMEM;
    memset(nep, 0, sizeof(*nep));
    nep->h = *h;
    nep->device = device;
    nep->stream = (cudaStream_t)cuda_stream;
    NepDims& d = nep->d;
    d.T = h->n_types; d.NR = h->n_max_radial + 1; d.KR = h->basis_radial + 1;
    d.NA = h->n_max_angular + 1; d.KA = h->basis_angular + 1;
    d.D = n_des(h); d.H = h->n_neurons;
    d.NRP = round_up4(d.NR); d.NAP = round_up4(d.NA); d.KRP = round_up4(d.KR);
    d.KAR = 1 + round_up4(d.KA - 1);
    d.has4 = h->l_max_4b >= 2; d.has5 = h->l_max_5b >= 1; d.nblk = 4 + d.has4 + d.has5;
    d.rcR = (float)h->rc_radial; d.rcA = (float)h->rc_angular;
    d.rcR_inv = (float)(1.0 / h->rc_radial); d.rcA_inv = (float)(1.0 / h->rc_angular);
    d.rcR2 = d.rcR * d.rcR; d.rcA2 = d.rcA * d.rcA;
    nep->DP = ann_tier(d.D);
    if (nep->DP < 0) { delete nep; return NEP_ERR_INVALID_ARG; }
    for (int t = 0; t < d.T; ++t) {
        if (!(mass_amu[t] > 0.0)) { delete nep; return NEP_ERR_INVALID_ARG; }
        nep->mass[t] = mass_amu[t];
    }

    // re-laid-out parameter tables (layouts documented at the kernels that read them)
    const int T = d.T, TT = T * T;
    nep->KP = round_up4(d.KR);
    nep->strideR = (d.KR * d.NRP) | 1;
    nep->nch_max = 5;
    bool nch_forced = false;
    nep->smem_budget = 180 * 1024;
    nep->ann_fp32 = getenv("NEP_ANN_FP32") != nullptr;                // tests / comparison: the fp32-FMA network kernel
    nep->force_smem_radial = getenv("NEP_RADIAL_SMEM") != nullptr;    // tests: exercise the shared-memory variants
    nep->raggedness = 1.0;
    if (const char* e = getenv("NEP_SMEM_KB")) { const int v = atoi(e); if (v >= 8 && v <= 227) nep->smem_budget = (size_t)v * 1024; }
    if (const char* e = getenv("NEP_NCH_MAX")) { const int v = atoi(e); if (v >= 1 && v <= NEP_NCH_MAX) { nep->nch_max = v; nch_forced = true; } }
    {   // angular passes: at most nch_max channels each, tables staged in shared memory; if a table would
        // not fit there, passes of 4 channels read it from global memory (zero-padded surplus channels)
        {
            cudaDeviceProp prop;
            if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaGetLastError(); delete nep; return NEP_ERR_CUDA; }
            nep->num_sms = prop.multiProcessorCount;
        }
        auto stride_of = [&](int nch) { return (d.KAR * round_up4(nch)) | 1; };
        // six or seven channels go in ONE pass (the descriptor kernel holds 24 x 7 sums in registers, the force
        // kernel keeps the G of channels 6-7 in shared memory); more channels in passes of at most nch_max
        if (!nch_forced && (d.NA == 6 || d.NA == 7)) nep->nch_max = d.NA;
        const int npass = (d.NA + nep->nch_max - 1) / nep->nch_max;
        const int base = d.NA / npass, rem = d.NA % npass;
        nep->angular_tab_smem = sizeof(float) * (size_t)TT * stride_of(base + (rem ? 1 : 0)) <= kSmemTableMax;
        int n0 = 0, off = 0;
        nep->n_pass = 0;
        while (n0 < d.NA) {
            const int p = nep->n_pass++;
            const int nch = nep->angular_tab_smem ? base + (p < rem ? 1 : 0) : 4;
            nep->pass_n0[p] = n0; nep->pass_nch[p] = nch; nep->pass_off[p] = off; nep->pass_stride[p] = stride_of(nch);
            off += TT * nep->pass_stride[p];
            n0 += nch;
        }
    }
    rc = upload_parameters(nep, c_radial, c_angular, w0, b0, w1, b1);
    if (rc != NEP_OK) { nep_destroy(nep); return rc; }
    {
        std::vector<double> vm(nep->mass, nep->mass + d.T);
        rc = dev_alloc(nep, &nep->mass_dev, vm.size());
        if (rc == NEP_OK && cudaMemcpy(nep->mass_dev, vm.data(), vm.size() * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess) rc = NEP_ERR_CUDA;
        if (rc != NEP_OK) { nep_destroy(nep); return rc; }
    }
    rc = dev_alloc(nep, &nep->flags, 8);
    if (rc == NEP_OK) rc = dev_alloc(nep, &nep->build_stat, 2);
    if (rc == NEP_OK) rc = dev_alloc(nep, &nep->tile_ctr, 64);
    if (rc == NEP_OK) rc = dev_alloc(nep, &nep->disp_max, 2);
    if (rc != NEP_OK) { nep_destroy(nep); return rc; }
    cudaMemset(nep->disp_max, 0, 2 * sizeof(unsigned));
    if (cudaDeviceSynchronize() != cudaSuccess) { nep_destroy(nep); return NEP_ERR_CUDA; }
    *out = nep;
    return NEP_OK;
}

int nep_destroy(nep_t* nep)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    cudaSetDevice(nep->device);
    cudaStreamSynchronize(nep->stream);
    for (int a = 0; a < nep->n_owned; ++a) cudaFree(nep->owned[a].p);
    if (nep->copy_stream) { cudaStreamDestroy(nep->copy_stream); cudaEventDestroy(nep->ev_pos); }
    if (nep->prof_ev) {
        for (int a = 0; a < 2 * NEP_PROF_PAIRS; ++a) cudaEventDestroy(nep->prof_ev[a]);
        free(nep->prof_ev);
        free(nep->prof_kid);
    }
    cudaGetLastError();
    delete nep;
    return NEP_OK;
}

int nep_neighbors(nep_t* nep, int64_t n, const double* pos_dev, const int32_t* type_dev, const double box[9], double skin)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!pos_dev || !type_dev) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer");
    NEP_CUDA(cudaSetDevice(nep->device));
    nep->have_lists = nep->have_eval = nep->force_current = false;
    NEP_TRY(setup_system(nep, n, box, skin));
    NEP_CUDA(cudaMemcpyAsync(nep->type_orig, type_dev, sizeof(int) * (size_t)n, cudaMemcpyDeviceToDevice, nep->stream));
    return build_lists(nep, pos_dev);
}

int nep_max_neighbors(nep_t* nep, int which, int32_t* max_count_host)
{
    if (!nep || !max_count_host || (which != 0 && which != 1)) return NEP_ERR_INVALID_ARG;
    if (!nep->have_lists) return nep_fail(nep, NEP_ERR_STATE, "nep_neighbors has not been called");
    *max_count_host = which == 0 ? nep->maxR_skin : nep->maxA_skin;
    return NEP_OK;
}

int nep_get_neighbors(nep_t* nep, int which, int32_t* count_dev, int32_t* list_dev, int32_t cap)
{
    if (!nep || !count_dev || !list_dev || (which != 0 && which != 1)) return NEP_ERR_INVALID_ARG;
    if (!nep->have_lists) return nep_fail(nep, NEP_ERR_STATE, "nep_neighbors has not been called");
    if (cap < (which == 0 ? nep->maxR_skin : nep->maxA_skin)) return nep_fail(nep, NEP_ERR_INVALID_ARG, "cap smaller than the longest list");
    NEP_CUDA(cudaSetDevice(nep->device));
    const int n = (int)nep->n;
    NEP_LAUNCH(NEP_K_EXPORT, k_export_lists<<<div_up(n, 128), 128, 0, nep->stream>>>(n, which, nep->perm, nep->listA, nep->cntA, nep->listS, nep->cntS,
                                                          count_dev, list_dev, cap));
    return NEP_OK;
}

int nep_get_last(nep_t* nep, double* energy_dev, double* force_dev, double* virial_dev)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!nep->have_eval) return nep_fail(nep, NEP_ERR_STATE, "no evaluation yet");
    NEP_CUDA(cudaSetDevice(nep->device));
    const size_t n = (size_t)nep->n;
    if (energy_dev) NEP_CUDA(cudaMemcpyAsync(energy_dev, nep->e_out, sizeof(double) * n, cudaMemcpyDeviceToDevice, nep->stream));
    if (force_dev) NEP_CUDA(cudaMemcpyAsync(force_dev, nep->f_out, sizeof(double) * 3 * n, cudaMemcpyDeviceToDevice, nep->stream));
    if (virial_dev) NEP_CUDA(cudaMemcpyAsync(virial_dev, nep->w_out, sizeof(double) * 9 * n, cudaMemcpyDeviceToDevice, nep->stream));
    return NEP_OK;
}

int nep_compute(nep_t* nep, const double* pos_dev, double* energy_dev, double* force_dev, double* virial_dev)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!pos_dev) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer");
    if (!nep->have_lists) return nep_fail(nep, NEP_ERR_STATE, "nep_neighbors has not been called");
    NEP_CUDA(cudaSetDevice(nep->device));
    NEP_TRY(evaluate(nep, pos_dev));
    nep->force_current = true;
    nep->force_pos_tag = pos_dev;
    return nep_get_last(nep, energy_dev, force_dev, virial_dev);
}

// thermostat of md_loop: none (NVE), Berendsen (reading A15) or Langevin (reading A16)
struct Thermostat {
    int kind;                 // 0 none, 1 Berendsen, 2 Langevin
    double t_start, t_stop, tau_fs;
    unsigned long long seed;
    int64_t first_step;
};

// pos_ready (optional): recorded on the stream as soon as the positions have their final values (after the
// drift of the last step), so that a copy on another stream can overlap the last force evaluation
// the lists are valid while no atom has moved more than skin/2 since the build (both atoms of a pair may approach)
static int skin_check(nep_t* nep, unsigned disp2_bits)
{
    float r2;
    memcpy(&r2, &disp2_bits, sizeof(r2));
    if (sqrt((double)r2) > 0.5 * nep->skin) {
        snprintf(nep->err, sizeof(nep->err), "an atom moved %.4g A since the last list build, more than skin/2 = %.4g A: pairs may have "
                 "been missed; use a smaller rebuild_every or a larger skin", sqrt((double)r2), 0.5 * nep->skin);
        return NEP_ERR_SKIN_EXCEEDED;
    }
    return NEP_OK;
}

// defer_check: the caller reads disp_max[1] itself after its own synchronisation (md_run_host)
static int md_loop(nep_t* nep, double* pos_dev, double* vel_dev, double dt_fs, int32_t n_steps, int32_t rebuild_every,
                   double skin, const Thermostat& th, cudaEvent_t pos_ready = nullptr, bool defer_check = false)
{
    unsigned disp_bits = 0;
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!pos_dev || !vel_dev || n_steps < 0 || rebuild_every < 1 || !(skin >= 0.0) || !(dt_fs == dt_fs))
        return nep_fail(nep, NEP_ERR_INVALID_ARG, "bad md_step argument");
    if (th.kind && (!(th.tau_fs > 0.0) || !(th.t_start >= 0.0) || !(th.t_stop >= 0.0)))
        return nep_fail(nep, NEP_ERR_INVALID_ARG, "bad thermostat argument");
    if (th.kind == 1 && th.tau_fs < dt_fs) return nep_fail(nep, NEP_ERR_INVALID_ARG, "Berendsen thermostat: tau_fs < dt_fs");
    if (!nep->have_lists) return nep_fail(nep, NEP_ERR_STATE, "nep_neighbors has not been called");
    NEP_CUDA(cudaSetDevice(nep->device));
    const int n = (int)nep->n;
    cudaStream_t st = nep->stream;
    if (skin != nep->skin) {
        // a different skin takes effect at once: lists are rebuilt for the current positions
        double box9[9];
        for (int a = 0; a < 9; ++a) box9[a] = nep->H[a];
        NEP_TRY(setup_system(nep, nep->n, box9, skin));
        NEP_TRY(build_lists(nep, pos_dev));
        nep->force_current = false;
    }
    if (!nep->force_current || nep->force_pos_tag != pos_dev) NEP_TRY(evaluate(nep, pos_dev));
    const double hdt = 0.5 * dt_fs * kAccConv;
    const int TB = 256;
    const int nb = div_up(n, 256);
    if (th.kind == 1 && nb + 2 > nep->thermo_cap) {
        nep->thermo_cap = 0;
        NEP_TRY(dev_alloc(nep, &nep->thermo, (size_t)nb + 2));
        nep->thermo_cap = nb + 2;
    }
    if (pos_ready && n_steps == 0) NEP_CUDA(cudaEventRecord(pos_ready, st));
    const double lc1 = th.kind == 2 ? exp(-dt_fs / (2.0 * th.tau_fs)) : 1.0, lc2 = sqrt(1.0 - lc1 * lc1);
    for (int s = 0; s < n_steps; ++s) {
        const double t_target = th.kind ? th.t_start + (th.t_stop - th.t_start) * (double)(s + 1) / (double)n_steps : 0.0;
        if (th.kind == 2)
            NEP_LAUNCH(NEP_K_THERMOSTAT, k_langevin_half<<<div_up(3 * (int64_t)n, TB), TB, 0, st>>>(n, lc1, lc2, kBoltzmann * t_target * kAccConv, th.seed,
                                                      2ull * (unsigned long long)(th.first_step + s), nep->type_orig, nep->mass_dev, vel_dev));
        // NVE: the closing half kick of step s - 1 is fused with the opening half kick + drift of step s
        const bool fuse_kicks = th.kind == 0;
        if (fuse_kicks && s > 0)
            NEP_LAUNCH(NEP_K_KICK_DRIFT, k_kick_kick_drift<<<div_up(3 * (int64_t)n, TB), TB, 0, st>>>(n, hdt, dt_fs, nep->type_orig, nep->mass_dev, nep->f_out, vel_dev, pos_dev));
        else
            NEP_LAUNCH(NEP_K_KICK_DRIFT, k_kick_drift<<<div_up(3 * (int64_t)n, TB), TB, 0, st>>>(n, hdt, dt_fs, nep->type_orig, nep->mass_dev, nep->f_out, vel_dev, pos_dev));
        if (pos_ready && s == n_steps - 1) NEP_CUDA(cudaEventRecord(pos_ready, st));
        nep->steps_since_build++;
        if (nep->steps_since_build >= rebuild_every) {
            // skin check of the interval that ends here, BEFORE the rebuild: &disp_bits is pageable memory, so the
            // copy has completed when the call returns; a run that lost pairs reports that, not whatever the
            // rebuild of the broken state would have returned, and does not pay for that rebuild
            NEP_CUDA(cudaMemcpyAsync(&disp_bits, nep->disp_max + 1, sizeof(unsigned), cudaMemcpyDeviceToHost, st));
            NEP_CUDA(cudaStreamSynchronize(st));
            NEP_TRY(skin_check(nep, disp_bits));
            NEP_TRY(build_lists(nep, pos_dev));
        }
        NEP_TRY(evaluate(nep, pos_dev));
        if (!fuse_kicks || s == n_steps - 1)
            NEP_LAUNCH(NEP_K_KICK, k_kick<<<div_up(3 * (int64_t)n, TB), TB, 0, st>>>(n, hdt, nep->type_orig, nep->mass_dev, nep->f_out, vel_dev));
        if (th.kind == 2)
            NEP_LAUNCH(NEP_K_THERMOSTAT, k_langevin_half<<<div_up(3 * (int64_t)n, TB), TB, 0, st>>>(n, lc1, lc2, kBoltzmann * t_target * kAccConv, th.seed,
                                                      2ull * (unsigned long long)(th.first_step + s) + 1ull, nep->type_orig, nep->mass_dev, vel_dev));
        if (th.kind == 1) {
            double* lam = nep->thermo + (nep->thermo_cap - 2);
            NEP_LAUNCH(NEP_K_THERMOSTAT, k_mv2_partial<<<nb, 256, 0, st>>>(n, nep->type_orig, nep->mass_dev, vel_dev, nep->thermo));
            NEP_LAUNCH(NEP_K_THERMOSTAT, k_berendsen_lambda<<<1, 256, 0, st>>>(nb, nep->thermo, 1.0 / (kAccConv * 3.0 * (double)n * kBoltzmann),
                                                                              dt_fs / th.tau_fs, t_target, lam));
            NEP_LAUNCH(NEP_K_THERMOSTAT, k_scale_velocities<<<div_up(3 * (int64_t)n, TB), TB, 0, st>>>(3 * n, lam, vel_dev));
        }
    }
    nep->force_current = true;
    nep->force_pos_tag = pos_dev;
    if (n_steps > 0 && !defer_check) {
        NEP_CUDA(cudaMemcpyAsync(&disp_bits, nep->disp_max + 1, sizeof(unsigned), cudaMemcpyDeviceToHost, st));
        NEP_CUDA(cudaStreamSynchronize(st));
        NEP_TRY(skin_check(nep, disp_bits));
    }
    return NEP_OK;
}

int md_step(nep_t* nep, double* pos_dev, double* vel_dev, double dt_fs, int32_t n_steps, int32_t rebuild_every, double skin)
{
    const Thermostat none = {0, 0.0, 0.0, 0.0, 0ull, 0};
    return md_loop(nep, pos_dev, vel_dev, dt_fs, n_steps, rebuild_every, skin, none);
}

int md_step_nvt_berendsen(nep_t* nep, double* pos_dev, double* vel_dev, double dt_fs, int32_t n_steps, int32_t rebuild_every,
                          double skin, double t_start_K, double t_stop_K, double tau_fs)
{
    const Thermostat th = {1, t_start_K, t_stop_K, tau_fs, 0ull, 0};
    return md_loop(nep, pos_dev, vel_dev, dt_fs, n_steps, rebuild_every, skin, th);
}

int md_step_nvt_langevin(nep_t* nep, double* pos_dev, double* vel_dev, double dt_fs, int32_t n_steps, int32_t rebuild_every,
                         double skin, double t_start_K, double t_stop_K, double tau_fs, uint64_t seed, int64_t first_step)
{
    if (first_step < 0) return nep_fail(nep, NEP_ERR_INVALID_ARG, "bad thermostat argument");
    const Thermostat th = {2, t_start_K, t_stop_K, tau_fs, (unsigned long long)seed, first_step};
    return md_loop(nep, pos_dev, vel_dev, dt_fs, n_steps, rebuild_every, skin, th);
}

int nep_last_temperature(nep_t* nep, double* t_before_host, double* lambda_host)
{
    if (!nep || (!t_before_host && !lambda_host)) return NEP_ERR_INVALID_ARG;
    if (!nep->thermo || nep->thermo_cap < 2) return nep_fail(nep, NEP_ERR_STATE, "no thermostatted step yet");
    NEP_CUDA(cudaSetDevice(nep->device));
    double v[2];
    NEP_CUDA(cudaMemcpyAsync(v, nep->thermo + (nep->thermo_cap - 2), sizeof(v), cudaMemcpyDeviceToHost, nep->stream));
    NEP_CUDA(cudaStreamSynchronize(nep->stream));
    if (lambda_host) *lambda_host = v[0];
    if (t_before_host) *t_before_host = v[1];
    return NEP_OK;
}

int nep_max_displacement(nep_t* nep, double* disp_host)
{
    if (!nep || !disp_host) return NEP_ERR_INVALID_ARG;
    if (!nep->have_eval) return nep_fail(nep, NEP_ERR_STATE, "no evaluation yet");
    NEP_CUDA(cudaSetDevice(nep->device));
    unsigned bits = 0;
    NEP_CUDA(cudaMemcpyAsync(&bits, nep->disp_max, sizeof(bits), cudaMemcpyDeviceToHost, nep->stream));
    NEP_CUDA(cudaStreamSynchronize(nep->stream));
    float r2;
    memcpy(&r2, &bits, sizeof(r2));
    *disp_host = sqrt((double)r2);
    return NEP_OK;
}

int nep_list_raggedness(nep_t* nep, double* raggedness_host)
{
    if (!nep || !raggedness_host) return NEP_ERR_INVALID_ARG;
    if (!nep->have_lists) return nep_fail(nep, NEP_ERR_STATE, "nep_neighbors has not been called");
    *raggedness_host = nep->raggedness;
    return NEP_OK;
}

int nep_get_descriptors(nep_t* nep, float* q_dev, float* fp_dev)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!nep->have_eval) return nep_fail(nep, NEP_ERR_STATE, "no evaluation yet");
    NEP_CUDA(cudaSetDevice(nep->device));
    const int n = (int)nep->n;
    if (q_dev) { NEP_LAUNCH(NEP_K_EXPORT, k_export_rows<<<div_up(n, 128), 128, 0, nep->stream>>>(n, nep->d.D, nep->perm, nep->q, q_dev)); }
    if (fp_dev) { NEP_LAUNCH(NEP_K_EXPORT, k_export_rows<<<div_up(n, 128), 128, 0, nep->stream>>>(n, nep->d.D, nep->perm, nep->fp, fp_dev)); }
    return NEP_OK;
}

int nep_get_angular_sums(nep_t* nep, float* S_dev)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!nep->have_eval) return nep_fail(nep, NEP_ERR_STATE, "no evaluation yet");
    NEP_CUDA(cudaSetDevice(nep->device));
    const int n = (int)nep->n;
    if (S_dev) { NEP_LAUNCH(NEP_K_EXPORT, k_export_rows<<<div_up(n, 128), 128, 0, nep->stream>>>(n, nep->d.NA * NEP_NUM_S, nep->perm, nep->S, S_dev)); }
    return NEP_OK;
}

// ---- derived outputs ----------------------------------------------------
int nep_set_parameters(nep_t* nep, const float* c_radial, const float* c_angular, const float* w0, const float* b0,
                       const float* w1, const float* b1)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!c_radial || !c_angular || !w0 || !b0 || !w1 || !b1) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer");
    NEP_CUDA(cudaSetDevice(nep->device));
    NEP_TRY(upload_parameters(nep, c_radial, c_angular, w0, b0, w1, b1));
    nep->have_eval = nep->force_current = false;         // E/F/W of the old model no longer apply
    return NEP_OK;
}

int nep_compute_population(nep_t* nep, const double* pos_dev, int32_t n_pop, const float* c_radial, const float* c_angular,
                           const float* w0, const float* b0, const float* w1, const float* b1,
                           double* energy_dev, double* force_dev, double* virial_dev)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!pos_dev || n_pop < 1 || !c_radial || !c_angular || !w0 || !b0 || !w1 || !b1) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer or n_pop < 1");
    if (!nep->have_lists) return nep_fail(nep, NEP_ERR_STATE, "nep_neighbors has not been called");
    NEP_CUDA(cudaSetDevice(nep->device));
    const NepDims& d = nep->d;
    const size_t n = (size_t)nep->n;
    const size_t sR = (size_t)d.T * d.T * d.NR * d.KR, sA = (size_t)d.T * d.T * d.NA * d.KA, sW = (size_t)d.H * d.D;
    for (int32_t m = 0; m < n_pop; ++m) {
        NEP_TRY(upload_parameters(nep, c_radial + m * sR, c_angular + m * sA, w0 + m * sW, b0 + (size_t)m * d.H, w1 + (size_t)m * d.H, b1 + m));
        // the geometry is the population's: positions are quantised and the lists filtered once
        NEP_TRY(evaluate(nep, pos_dev, m > 0));
        NEP_TRY(nep_get_last(nep, energy_dev ? energy_dev + m * n : nullptr, force_dev ? force_dev + 3 * m * n : nullptr,
                             virial_dev ? virial_dev + 9 * m * n : nullptr));
    }
    nep->force_current = false;                          // the handle now holds the LAST member's model and forces
    return NEP_OK;
}

int nep_loss_terms(nep_t* nep, double u_target_per_atom, const double* f_target_dev, const double w_target_per_atom[6],
                   double terms_host[3])
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!f_target_dev || !w_target_per_atom || !terms_host) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer");
    if (!nep->have_eval) return nep_fail(nep, NEP_ERR_STATE, "no evaluation yet");
    NEP_CUDA(cudaSetDevice(nep->device));
    const int n = (int)nep->n;
    const int nb = div_up(n, 256);
    if (11 * nb + 11 > nep->loss_cap) {
        nep->loss_cap = 0;
        NEP_TRY(dev_alloc(nep, &nep->loss_partial, 11 * (size_t)nb + 11));
        nep->loss_cap = 11 * nb + 11;
    }
    double* tot_dev = nep->loss_partial + 11 * (size_t)nb;
    NEP_LAUNCH(NEP_K_EXPORT, k_loss_partial<<<nb, 256, 0, nep->stream>>>(n, nep->e_out, nep->f_out, nep->w_out, f_target_dev, nep->loss_partial));
    NEP_LAUNCH(NEP_K_EXPORT, k_loss_total<<<1, 256, 0, nep->stream>>>(nb, nep->loss_partial, tot_dev));
    double t[11];
    NEP_CUDA(cudaMemcpyAsync(t, tot_dev, sizeof(t), cudaMemcpyDeviceToHost, nep->stream));
    NEP_CUDA(cudaStreamSynchronize(nep->stream));
    const double N = (double)n;
    terms_host[0] = fabs(t[0] / N - u_target_per_atom);
    terms_host[1] = sqrt(t[1] / (3.0 * N));
    const int six[6] = {0, 4, 8, 1, 5, 6};               // xx, yy, zz, xy, yz, zx of W[3a+b]
    double sv = 0.0;
    for (int c = 0; c < 6; ++c) { const double dv = t[2 + six[c]] / N - w_target_per_atom[c]; sv += dv * dv; }
    terms_host[2] = sqrt(sv / 6.0);
    return NEP_OK;
}

int nep_get_latent(nep_t* nep, float* latent_dev)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!latent_dev) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer");
    if (!nep->have_eval) return nep_fail(nep, NEP_ERR_STATE, "no evaluation yet");
    NEP_CUDA(cudaSetDevice(nep->device));
    switch (nep->DP) {
        case 24: return launch_latent<24>(nep, latent_dev);
        case 40: return launch_latent<40>(nep, latent_dev);
        case 56: return launch_latent<56>(nep, latent_dev);
        case 72: return launch_latent<72>(nep, latent_dev);
        case 88: return launch_latent<88>(nep, latent_dev);
        case 104: return launch_latent<104>(nep, latent_dev);
        case 120: return launch_latent<120>(nep, latent_dev);
    }
    return nep_fail(nep, NEP_ERR_INVALID_ARG, "descriptor too long");
}

int nep_heat_current(nep_t* nep, const double* vel_dev, double* j_atom_dev, double* j_total_dev)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!vel_dev || (!j_atom_dev && !j_total_dev)) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer");
    if (!nep->have_eval) return nep_fail(nep, NEP_ERR_STATE, "no evaluation yet");
    NEP_CUDA(cudaSetDevice(nep->device));
    const int n = (int)nep->n;
    const int nb = div_up(n, 256);
    if (nb > nep->heat_cap) {
        nep->heat_cap = 0;
        NEP_TRY(dev_alloc(nep, &nep->heat_partial, 3 * (size_t)nb + 3));
        nep->heat_cap = nb;
    }
    NEP_LAUNCH(NEP_K_EXPORT, k_heat_current<<<nb, 256, 0, nep->stream>>>(n, nep->w_out, vel_dev, j_atom_dev, nep->heat_partial));
    double* tot = j_total_dev ? j_total_dev : nep->heat_partial + 3 * (size_t)nb;
    NEP_LAUNCH(NEP_K_EXPORT, k_heat_total<<<1, 256, 0, nep->stream>>>(nb, nep->heat_partial, tot));
    return NEP_OK;
}

// ---- heat current without any allocation (nep_heat_current_static, include/nep.h) ------------------------
// nep_heat_current keeps its block partials in a cudaMalloc'ed buffer that grows with the system.  Some users
// of this library sample J every few steps from places where a device allocation is not an option: a Green-Kubo
// production loop that has handed all free device memory to another allocator (PyTorch's caching allocator,
// a second simulation on the same GPU), where cudaMalloc fails although the 400 kB are trivially "there"; or a
// latency-sensitive service thread, for which the device-wide synchronisation that cudaMalloc / cudaFree may
// imply stalls every other stream of the process.  For them the partials live in the array below, which is part
// of the library image: every GPU that loads libnep_b200.so carries these 393,240 bytes from the first CUDA call
// to process exit, whether or not the entry point is ever used.
//
// g_heat_static is a DEVICE symbol.  In host code its name is only a host-side shadow of it: handing
// `g_heat_static` itself to a kernel would pass a host address (a fault, or on systems where the GPU can reach host
// memory a silent write to the wrong place).  The device address comes from cudaGetSymbolAddress, asked once per
// device with that device current (heat_static_address), and that pointer is what the kernels receive.
#define NEP_HEAT_STATIC_MAX_ATOMS 4194304                       /* stated limit of the entry point           */
#define NEP_HEAT_STATIC_MAX_BLOCKS (NEP_HEAT_STATIC_MAX_ATOMS / 256)
#define NEP_HEAT_STATIC_MAX_DEVICES 64
static __device__ __align__(256) double g_heat_static[3 * NEP_HEAT_STATIC_MAX_BLOCKS + 3];

namespace {
std::mutex g_heat_static_mutex;
double* g_heat_static_ptr[NEP_HEAT_STATIC_MAX_DEVICES];         // device address of g_heat_static, per device

// Device address of g_heat_static on `device`, which must be the current device.  The first call per device asks
// the runtime (no allocation: the array was placed when the module was loaded); later calls read the table.
cudaError_t heat_static_address(int device, double** out)
{
    std::lock_guard<std::mutex> lock(g_heat_static_mutex);
    if (!g_heat_static_ptr[device]) {
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_heat_static);
        if (e != cudaSuccess) return e;
        g_heat_static_ptr[device] = p;
    }
    *out = g_heat_static_ptr[device];
    return cudaSuccess;
}
}  // namespace

int nep_heat_current_static(nep_t* nep, const double* vel_dev, double* j_atom_dev, double* j_total_dev)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!vel_dev || (!j_atom_dev && !j_total_dev)) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer");
    if (!nep->have_eval) return nep_fail(nep, NEP_ERR_STATE, "no evaluation yet");
    if (nep->n > NEP_HEAT_STATIC_MAX_ATOMS) {
        snprintf(nep->err, sizeof(nep->err),
                 "nep_heat_current_static: %lld atoms exceed the static scratch's limit of %d atoms; use nep_heat_current",
                 (long long)nep->n, NEP_HEAT_STATIC_MAX_ATOMS);
        return NEP_ERR_INVALID_ARG;
    }
    if (nep->device < 0 || nep->device >= NEP_HEAT_STATIC_MAX_DEVICES)
        return nep_fail(nep, NEP_ERR_INVALID_ARG, "nep_heat_current_static: device ordinal beyond the per-device table (64)");
    NEP_CUDA(cudaSetDevice(nep->device));
    double* scratch = nullptr;
    NEP_CUDA(heat_static_address(nep->device, &scratch));
    const int n = (int)nep->n;
    const int nb = div_up(n, 256);
    // Nothing has to start at zero: each of the nb blocks stores its three partials unconditionally, and the
    // second kernel (same stream, so after the first) reads exactly those 3 nb values.  Whatever an earlier
    // call left beyond them is never read.  Plain launches: the profiling hooks of NEP_LAUNCH are left out.
    k_heat_current<<<nb, 256, 0, nep->stream>>>(n, nep->w_out, vel_dev, j_atom_dev, scratch);
    NEP_LAUNCH_CHECK();
    double* tot = j_total_dev ? j_total_dev : scratch + 3 * (size_t)NEP_HEAT_STATIC_MAX_BLOCKS;
    k_heat_total<<<1, 256, 0, nep->stream>>>(nb, scratch, tot);
    NEP_LAUNCH_CHECK();
    return NEP_OK;
}

// ---- batched evaluation for training (nep_batch.cuh) --------------------------
int nep_batch_neighbors(nep_t* nep, int32_t n_str, const int32_t* atom_offset_host, const double* pos_dev,
                        const int32_t* type_dev, const double* boxes_host)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (n_str < 1 || !atom_offset_host || !pos_dev || !type_dev || !boxes_host) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer or n_str < 1");
    if (atom_offset_host[0] != 0) return nep_fail(nep, NEP_ERR_INVALID_ARG, "atom_offset[0] must be 0");
    for (int s = 0; s < n_str; ++s)
        if (atom_offset_host[s + 1] <= atom_offset_host[s]) return nep_fail(nep, NEP_ERR_INVALID_ARG, "every structure needs at least one atom");
    NEP_CUDA(cudaSetDevice(nep->device));
    const int N = atom_offset_host[n_str];
    std::vector<double> H(9 * (size_t)n_str), Hinv(9 * (size_t)n_str);
    std::vector<int> M(3 * (size_t)n_str), sid((size_t)N);
    for (int s = 0; s < n_str; ++s) {
        const double* h = boxes_host + 9 * (size_t)s;
        for (int a = 0; a < 9; ++a)
            if (!(h[a] == h[a]) || fabs(h[a]) > 1e12) return nep_fail(nep, NEP_ERR_INVALID_ARG, "bad box");
        const double c00 = h[4] * h[8] - h[5] * h[7], c01 = h[5] * h[6] - h[3] * h[8], c02 = h[3] * h[7] - h[4] * h[6];
        const double det = (h[0] * c00 + h[1] * c01) + h[2] * c02;
        if (!(det > 0.0)) return nep_fail(nep, NEP_ERR_UNSUPPORTED_BOX, "the cell vectors a, b, c must form a right-handed, non-degenerate cell");
        double* inv = Hinv.data() + 9 * (size_t)s;
        inv[0] = c00 / det; inv[1] = (h[2] * h[7] - h[1] * h[8]) / det; inv[2] = (h[1] * h[5] - h[2] * h[4]) / det;
        inv[3] = c01 / det; inv[4] = (h[0] * h[8] - h[2] * h[6]) / det; inv[5] = (h[2] * h[3] - h[0] * h[5]) / det;
        inv[6] = c02 / det; inv[7] = (h[1] * h[6] - h[0] * h[7]) / det; inv[8] = (h[0] * h[4] - h[1] * h[3]) / det;
        for (int k = 0; k < 3; ++k) {
            const double width = 1.0 / sqrt(inv[k] * inv[k] + inv[3 + k] * inv[3 + k] + inv[6 + k] * inv[6 + k]);
            const int m = (int)floor(nep->h.rc_radial / width + 0.5) + 1;       // reading A18
            if (m > NEP_BATCH_MAX_SHIFT) return nep_fail(nep, NEP_ERR_BOX_TOO_SMALL, "a cell of the batch is thinner than rc_radial / 6.5");
            M[3 * (size_t)s + k] = m;
        }
        for (int a = 0; a < 9; ++a) H[9 * (size_t)s + a] = h[a];
        for (int i = atom_offset_host[s]; i < atom_offset_host[s + 1]; ++i) sid[(size_t)i] = s;
    }
    auto& b = nep->b;
    b.n_str = 0;                                          // invalid until everything below succeeds
    NEP_TRY(dev_alloc(nep, &b.off, (size_t)n_str + 1));
    NEP_TRY(dev_alloc(nep, &b.sid, (size_t)N));
    NEP_TRY(dev_alloc(nep, &b.M, 3 * (size_t)n_str));
    NEP_TRY(dev_alloc(nep, &b.H, 9 * (size_t)n_str));
    NEP_TRY(dev_alloc(nep, &b.Hinv, 9 * (size_t)n_str));
    NEP_TRY(dev_alloc(nep, &b.type, (size_t)N));
    NEP_TRY(dev_alloc(nep, &b.cnt, (size_t)N));
    NEP_TRY(dev_alloc(nep, &b.cntA, (size_t)N));
    if (!b.bad) NEP_TRY(dev_alloc(nep, &b.bad, 1));
    cudaStream_t st = nep->stream;
    NEP_CUDA(cudaMemcpyAsync(b.off, atom_offset_host, sizeof(int) * ((size_t)n_str + 1), cudaMemcpyHostToDevice, st));
    NEP_CUDA(cudaMemcpyAsync(b.sid, sid.data(), sizeof(int) * (size_t)N, cudaMemcpyHostToDevice, st));
    NEP_CUDA(cudaMemcpyAsync(b.M, M.data(), sizeof(int) * M.size(), cudaMemcpyHostToDevice, st));
    NEP_CUDA(cudaMemcpyAsync(b.H, H.data(), sizeof(double) * H.size(), cudaMemcpyHostToDevice, st));
    NEP_CUDA(cudaMemcpyAsync(b.Hinv, Hinv.data(), sizeof(double) * Hinv.size(), cudaMemcpyHostToDevice, st));
    NEP_CUDA(cudaMemcpyAsync(b.type, type_dev, sizeof(int) * (size_t)N, cudaMemcpyDeviceToDevice, st));
    NEP_CUDA(cudaMemsetAsync(b.bad, 0, sizeof(int), st));
    // count, size the storage from the longest list, fill, reverse slots
    NEP_LAUNCH(NEP_K_BATCH, kb_neighbors<<<div_up(N, 128), 128, 0, st>>>(N, b.sid, b.off, b.H, b.Hinv, b.M, pos_dev, b.type, nep->d.T, nep->h.rc_radial, nep->d.rcA, 0, 0,
                                                                          b.cnt, b.cntA, nullptr, nullptr, nullptr, nullptr, b.bad));
    std::vector<int> cnt((size_t)N);
    int bad = 0;
    NEP_CUDA(cudaMemcpyAsync(cnt.data(), b.cnt, sizeof(int) * (size_t)N, cudaMemcpyDeviceToHost, st));
    NEP_CUDA(cudaMemcpyAsync(&bad, b.bad, sizeof(int), cudaMemcpyDeviceToHost, st));
    NEP_CUDA(cudaStreamSynchronize(st));                  // the host vectors above are temporaries, too
    if (bad & 2) return nep_fail(nep, NEP_ERR_INVALID_ARG, "an atom type is outside [0, n_types)");
    int cap = 1;
    for (int i = 0; i < N; ++i) if (cnt[(size_t)i] > cap) cap = cnt[(size_t)i];
    if (cap > 65535) return nep_fail(nep, NEP_ERR_NEIGHBOR_OVERFLOW, "more than 65535 neighbour entries per atom");
    NEP_TRY(dev_alloc(nep, &b.nbr, (size_t)N * cap));
    NEP_TRY(dev_alloc(nep, &b.d, (size_t)N * cap));
    NEP_TRY(dev_alloc(nep, &b.code, (size_t)N * cap));
    NEP_TRY(dev_alloc(nep, &b.tnb, (size_t)N * cap));
    NEP_TRY(dev_alloc(nep, &b.rev, (size_t)N * cap));
    NEP_LAUNCH(NEP_K_BATCH, kb_neighbors<<<div_up(N, 128), 128, 0, st>>>(N, b.sid, b.off, b.H, b.Hinv, b.M, pos_dev, b.type, nep->d.T, nep->h.rc_radial, nep->d.rcA, 1, cap,
                                                                          b.cnt, b.cntA, b.nbr, b.d, b.code, b.tnb, b.bad));
    NEP_LAUNCH(NEP_K_BATCH, kb_reverse<<<div_up(N, 128), 128, 0, st>>>(N, cap, b.cnt, b.nbr, b.code, b.rev, b.bad));
    NEP_CUDA(cudaMemcpyAsync(&bad, b.bad, sizeof(int), cudaMemcpyDeviceToHost, st));
    NEP_CUDA(cudaStreamSynchronize(st));
    if (bad & 1) return nep_fail(nep, NEP_ERR_CUDA, "batch neighbours: an entry has no reverse entry (internal error)");
    b.N = N; b.cap = cap; b.n_str = n_str; b.scratch_rows = 0;
    return NEP_OK;
}

int nep_batch_compute(nep_t* nep, int32_t n_pop, const float* c_radial, const float* c_angular, const float* w0, const float* b0,
                      const float* w1, const float* b1, double* energy_dev, double* force_dev, double* virial_dev)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (n_pop < 1 || !c_radial || !c_angular || !w0 || !b0 || !w1 || !b1 || !energy_dev) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer or n_pop < 1");
    auto& b = nep->b;
    if (b.n_str < 1) return nep_fail(nep, NEP_ERR_STATE, "nep_batch_neighbors has not been called");
    NEP_CUDA(cudaSetDevice(nep->device));
    static const NepCoef C = make_coef();
    const NepDims& d = nep->d;
    cudaStream_t st = nep->stream;
    const size_t N = (size_t)b.N;
    // parameters of ALL members: six copies, no per-member synchronisation
    const size_t per[6] = {(size_t)d.T * d.T * d.NR * d.KR, (size_t)d.T * d.T * d.NA * d.KA, (size_t)d.H * d.D, (size_t)d.H, (size_t)d.H, 1};
    const float* src[6] = {c_radial, c_angular, w0, b0, w1, b1};
    for (int a = 0; a < 6; ++a) {
        if (per[a] * n_pop > b.par_cap[a]) {
            b.par_cap[a] = 0;
            NEP_TRY(dev_alloc(nep, &b.par[a], per[a] * n_pop));
            b.par_cap[a] = per[a] * n_pop;
        }
        NEP_CUDA(cudaMemcpyAsync(b.par[a], src[a], sizeof(float) * per[a] * n_pop, cudaMemcpyHostToDevice, st));
    }
    // scratch per (member, atom); members in chunks of at most ~4 GB
    const size_t row_bytes = sizeof(float) * (2 * (size_t)d.D + (size_t)d.NA * NEP_NUM_S) + sizeof(float4) * b.cap;
    size_t mchunk = (size_t)4e9 / (row_bytes * N);
    if (mchunk < 1) mchunk = 1;
    if (mchunk > (size_t)n_pop) mchunk = (size_t)n_pop;
    if (mchunk > 65535) mchunk = 65535;                  // gridDim.y
    if (mchunk * N > b.scratch_rows) {
        b.scratch_rows = 0;
        NEP_TRY(dev_alloc(nep, &b.q, mchunk * N * d.D));
        NEP_TRY(dev_alloc(nep, &b.fp, mchunk * N * d.D));
        NEP_TRY(dev_alloc(nep, &b.S, mchunk * N * d.NA * NEP_NUM_S));
        NEP_TRY(dev_alloc(nep, &b.pf, mchunk * N * b.cap));
        b.scratch_rows = mchunk * N;
    }
    for (size_t p0 = 0; p0 < (size_t)n_pop; p0 += mchunk) {
        const int np = (int)((size_t)n_pop - p0 < mchunk ? (size_t)n_pop - p0 : mchunk);
        BatchParams P = {b.par[0] + p0 * per[0], b.par[1] + p0 * per[1], b.par[2] + p0 * per[2], b.par[3] + p0 * per[3],
                         b.par[4] + p0 * per[4], b.par[5] + p0 * per[5]};
        const dim3 grid(div_up(b.N, 128), np);
        // angular channels per pass: all of them for five to seven channels (one pass), else four at a time
#define NEP_KB_LAUNCH(NCHB)                                                                                     \
        do {                                                                                                    \
            int bs = 128;                                 /* per-thread sums / E table + the pass's coefficient table */ \
            auto smem = [&](int b_) { return sizeof(float) * ((size_t)d.T * d.KR * b_ + (size_t)d.T * d.T * d.KA * NCHB); }; \
            while (bs > 32 && smem(bs) > 100 * 1024) bs >>= 1;                                                   \
            if (smem(bs) > 200 * 1024) return nep_fail(nep, NEP_ERR_INVALID_ARG, "n_types x basis too large for shared memory"); \
            const dim3 gridb(div_up(b.N, bs), np);                                                               \
            NEP_TRY(allow_smem(nep, kb_descriptors<NCHB>, smem(bs)));                                            \
            NEP_TRY(allow_smem(nep, kb_partial<NCHB>, smem(bs)));                                                \
            NEP_LAUNCH(NEP_K_BATCH_DESC, kb_descriptors<NCHB><<<gridb, bs, smem(bs), st>>>(d, C, b.N, b.cap, P, b.type, b.cnt, b.tnb, b.d, b.q, b.S, b.cntA)); \
            NEP_TRY(launch_batch_ann(nep, grid, P, energy_dev + p0 * N));                                       \
            if (force_dev || virial_dev)                                                                        \
                NEP_LAUNCH(NEP_K_BATCH_PARTIAL, kb_partial<NCHB><<<gridb, bs, smem(bs), st>>>(d, C, b.N, b.cap, P, b.type, b.cnt, b.tnb, b.d, b.S, b.fp, b.pf, b.cntA)); \
        } while (0)
        switch (d.NA) {
            case 5: NEP_KB_LAUNCH(5); break;
            case 6: NEP_KB_LAUNCH(6); break;
            case 7: NEP_KB_LAUNCH(7); break;
            default: NEP_KB_LAUNCH(4); break;
        }
#undef NEP_KB_LAUNCH
        if (force_dev || virial_dev) {
            NEP_LAUNCH(NEP_K_BATCH_GATHER, kb_gather<<<grid, 128, 0, st>>>(b.N, b.cap, b.cnt, b.nbr, b.d, b.rev, b.pf, force_dev ? force_dev + 3 * p0 * N : nullptr,
                                                                    virial_dev ? virial_dev + 9 * p0 * N : nullptr));
        }
    }
    NEP_CUDA(cudaStreamSynchronize(st));                  // the caller may free or reuse its host parameter arrays
    return NEP_OK;
}

int nep_batch_pair_counts(nep_t* nep, int64_t* radial_entries_host, int64_t* angular_entries_host)
{
    if (!nep || !radial_entries_host || !angular_entries_host) return NEP_ERR_INVALID_ARG;
    auto& b = nep->b;
    if (b.n_str < 1) return nep_fail(nep, NEP_ERR_STATE, "nep_batch_neighbors has not been called");
    NEP_CUDA(cudaSetDevice(nep->device));
    std::vector<int> c((size_t)b.N), ca((size_t)b.N);
    NEP_CUDA(cudaMemcpyAsync(c.data(), b.cnt, sizeof(int) * (size_t)b.N, cudaMemcpyDeviceToHost, nep->stream));
    NEP_CUDA(cudaMemcpyAsync(ca.data(), b.cntA, sizeof(int) * (size_t)b.N, cudaMemcpyDeviceToHost, nep->stream));
    NEP_CUDA(cudaStreamSynchronize(nep->stream));
    int64_t sr = 0, sa = 0;
    for (int i = 0; i < b.N; ++i) { sr += c[(size_t)i]; sa += ca[(size_t)i]; }
    *radial_entries_host = sr;
    *angular_entries_host = sa;
    return NEP_OK;
}

int nep_batch_loss(nep_t* nep, int32_t n_pop, const double* energy_dev, const double* force_dev, const double* virial_dev,
                   const double* u_target_dev, const double* f_target_dev, const double* w_target_dev, double* loss_dev)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (n_pop < 1 || !energy_dev || !force_dev || !virial_dev || !u_target_dev || !f_target_dev || !w_target_dev || !loss_dev)
        return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer or n_pop < 1");
    auto& b = nep->b;
    if (b.n_str < 1) return nep_fail(nep, NEP_ERR_STATE, "nep_batch_neighbors has not been called");
    NEP_CUDA(cudaSetDevice(nep->device));
    const size_t need = 3 * (size_t)n_pop * b.n_str;
    if (need > b.loss_cap) {
        b.loss_cap = 0;
        NEP_TRY(dev_alloc(nep, &b.loss_part, need));
        b.loss_cap = need;
    }
    for (int p0 = 0; p0 < n_pop; p0 += 65535) {
        const int np = n_pop - p0 < 65535 ? n_pop - p0 : 65535;
        const size_t o = (size_t)p0 * b.N;
        NEP_LAUNCH(NEP_K_BATCH_LOSS, kb_loss_partial<<<dim3(b.n_str, np), 128, 0, nep->stream>>>(b.N, b.n_str, b.off, energy_dev + o, force_dev + 3 * o, virial_dev + 9 * o,
                                                                                          u_target_dev, f_target_dev, w_target_dev, b.loss_part + 3 * (size_t)p0 * b.n_str));
    }
    NEP_LAUNCH(NEP_K_BATCH_LOSS, kb_loss_total<<<n_pop, 128, 0, nep->stream>>>(b.N, b.n_str, b.loss_part, loss_dev));
    return NEP_OK;
}

// ---- host-buffer entry points ---------------------------------------------------------------------------
static int stage_alloc(nep_t* nep, int64_t n)
{
    if (n <= nep->h_cap && nep->h_pos) return NEP_OK;
    nep->h_cap = 0;
    NEP_TRY(dev_alloc(nep, &nep->h_pos, 3 * (size_t)n));
    NEP_TRY(dev_alloc(nep, &nep->h_vel, 3 * (size_t)n));
    NEP_TRY(dev_alloc(nep, &nep->h_type, (size_t)n));
    nep->h_cap = n;
    return NEP_OK;
}

static int download_results(nep_t* nep, double* energy_host, double* force_host, double* virial_host)
{
    const size_t n = (size_t)nep->n;
    if (energy_host) NEP_CUDA(cudaMemcpyAsync(energy_host, nep->e_out, sizeof(double) * n, cudaMemcpyDeviceToHost, nep->stream));
    if (force_host) NEP_CUDA(cudaMemcpyAsync(force_host, nep->f_out, sizeof(double) * 3 * n, cudaMemcpyDeviceToHost, nep->stream));
    if (virial_host) NEP_CUDA(cudaMemcpyAsync(virial_host, nep->w_out, sizeof(double) * 9 * n, cudaMemcpyDeviceToHost, nep->stream));
    return NEP_OK;
}

int nep_compute_host(nep_t* nep, int64_t n, const double* pos_host, const int32_t* type_host, const double box[9],
                     double skin, double* energy_host, double* force_host, double* virial_host)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!pos_host || !type_host || n <= 0 || n > NEP_MAX_ATOMS) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer or bad n");
    NEP_CUDA(cudaSetDevice(nep->device));
    nep->h_run = false;
    NEP_TRY(stage_alloc(nep, n));
    NEP_CUDA(cudaMemcpyAsync(nep->h_pos, pos_host, sizeof(double) * 3 * (size_t)n, cudaMemcpyHostToDevice, nep->stream));
    NEP_CUDA(cudaMemcpyAsync(nep->h_type, type_host, sizeof(int) * (size_t)n, cudaMemcpyHostToDevice, nep->stream));
    NEP_TRY(nep_neighbors(nep, n, nep->h_pos, nep->h_type, box, skin));
    NEP_TRY(evaluate(nep, nep->h_pos));
    NEP_TRY(download_results(nep, energy_host, force_host, virial_host));
    NEP_CUDA(cudaStreamSynchronize(nep->stream));
    return NEP_OK;
}

int md_run_host(nep_t* nep, int64_t n, double* pos_host, double* vel_host, const int32_t* type_host, const double box[9],
                double dt_fs, int32_t n_steps, int32_t rebuild_every, double skin,
                double* energy_host, double* force_host, double* virial_host)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    if (!pos_host || !vel_host || n <= 0 || n > NEP_MAX_ATOMS) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null pointer or bad n");
    NEP_CUDA(cudaSetDevice(nep->device));
    const bool cont = (type_host == nullptr);
    if (cont && !(nep->h_run && n == nep->n && nep->have_lists))
        return nep_fail(nep, NEP_ERR_STATE, "md_run_host: type_host == NULL continues a run, but none is in progress for this n");
    if (!cont && !box) return nep_fail(nep, NEP_ERR_INVALID_ARG, "null box");
    nep->h_run = false;
    NEP_TRY(stage_alloc(nep, n));
    const size_t b3 = sizeof(double) * 3 * (size_t)n;
    NEP_CUDA(cudaMemcpyAsync(nep->h_pos, pos_host, b3, cudaMemcpyHostToDevice, nep->stream));
    NEP_CUDA(cudaMemcpyAsync(nep->h_vel, vel_host, b3, cudaMemcpyHostToDevice, nep->stream));
    if (!cont) {
        NEP_CUDA(cudaMemcpyAsync(nep->h_type, type_host, sizeof(int) * (size_t)n, cudaMemcpyHostToDevice, nep->stream));
        NEP_TRY(nep_neighbors(nep, n, nep->h_pos, nep->h_type, box, skin));
    }
    if (!nep->copy_stream) {
        NEP_CUDA(cudaStreamCreateWithFlags(&nep->copy_stream, cudaStreamNonBlocking));
        NEP_CUDA(cudaEventCreateWithFlags(&nep->ev_pos, cudaEventDisableTiming));
    }
    // the positions are final after the last drift: their download (on a second stream) overlaps the last
    // force evaluation; velocities, energies and forces follow on the compute stream
    const Thermostat none = {0, 0.0, 0.0, 0.0, 0ull, 0};
    NEP_TRY(md_loop(nep, nep->h_pos, nep->h_vel, dt_fs, n_steps, rebuild_every, skin, none, nep->ev_pos, true));
    unsigned disp_bits = 0;
    NEP_CUDA(cudaStreamWaitEvent(nep->copy_stream, nep->ev_pos, 0));
    NEP_CUDA(cudaMemcpyAsync(pos_host, nep->h_pos, b3, cudaMemcpyDeviceToHost, nep->copy_stream));
    NEP_CUDA(cudaMemcpyAsync(vel_host, nep->h_vel, b3, cudaMemcpyDeviceToHost, nep->stream));
    NEP_TRY(download_results(nep, energy_host, force_host, virial_host));
    // last: &disp_bits is pageable memory, so this copy returns only when the stream has reached it -- enqueued
    // before the downloads above it would hold the host back and the position download would no longer overlap
    // the force evaluation
    NEP_CUDA(cudaMemcpyAsync(&disp_bits, nep->disp_max + 1, sizeof(unsigned), cudaMemcpyDeviceToHost, nep->stream));
    NEP_CUDA(cudaStreamSynchronize(nep->stream));
    NEP_CUDA(cudaStreamSynchronize(nep->copy_stream));
    nep->h_run = true;
    return skin_check(nep, disp_bits);
}

// ---- measurement support ----------------------------------------------------------------------------------
static const char* const kKernelNames[NEP_K_COUNT] = {
    "cell_hist", "scan", "scatter", "sort_cells", "quantize", "build_lists", "build_rev", "filter", "radial",
    "angular", "ann", "force_angular", "force_radial", "final", "kick_drift", "kick", "thermostat", "export", "batch_neighbors",
    "batch_descriptors", "batch_ann", "batch_partial", "batch_gather", "batch_loss"};

int nep_profile_num_kernels(void) { return NEP_K_COUNT; }

const char* nep_profile_kernel_name(int k) { return (k >= 0 && k < NEP_K_COUNT) ? kKernelNames[k] : ""; }

int nep_profile(nep_t* nep, int enable)
{
    if (!nep) return NEP_ERR_INVALID_ARG;
    NEP_CUDA(cudaSetDevice(nep->device));
    if (enable && !nep->prof_ev) {
        nep->prof_ev = (cudaEvent_t*)calloc(2 * NEP_PROF_PAIRS, sizeof(cudaEvent_t));
        nep->prof_kid = (int*)calloc(NEP_PROF_PAIRS, sizeof(int));
        if (!nep->prof_ev || !nep->prof_kid) return nep_fail(nep, NEP_ERR_NOMEM, "profile buffers");
        for (int a = 0; a < 2 * NEP_PROF_PAIRS; ++a) NEP_CUDA(cudaEventCreate(&nep->prof_ev[a]));
    }
    nep_prof_drain(nep);
    for (int k = 0; k < NEP_K_COUNT; ++k) { nep->prof_ms[k] = 0.0; nep->prof_n[k] = 0; }
    nep->prof_on = enable != 0;
    return NEP_OK;
}

int nep_profile_read(nep_t* nep, double* ms_total_host, int64_t* launches_host)
{
    if (!nep || !ms_total_host || !launches_host) return NEP_ERR_INVALID_ARG;
    NEP_CUDA(cudaSetDevice(nep->device));
    nep_prof_drain(nep);
    for (int k = 0; k < NEP_K_COUNT; ++k) { ms_total_host[k] = nep->prof_ms[k]; launches_host[k] = nep->prof_n[k]; }
    return NEP_OK;
}

int nep_pair_counts(nep_t* nep, int64_t* radial_pairs_host, int64_t* angular_pairs_host)
{
    if (!nep || !radial_pairs_host || !angular_pairs_host) return NEP_ERR_INVALID_ARG;
    if (!nep->have_eval) return nep_fail(nep, NEP_ERR_STATE, "no evaluation yet");
    NEP_CUDA(cudaSetDevice(nep->device));
    const size_t n = (size_t)nep->n;
    std::vector<int> a(n), b(n);
    NEP_CUDA(cudaMemcpyAsync(a.data(), nep->ncA, sizeof(int) * n, cudaMemcpyDeviceToHost, nep->stream));
    NEP_CUDA(cudaMemcpyAsync(b.data(), nep->ncB, sizeof(int) * n, cudaMemcpyDeviceToHost, nep->stream));
    NEP_CUDA(cudaStreamSynchronize(nep->stream));
    int64_t sa = 0, sb = 0;
    for (size_t i = 0; i < n; ++i) { sa += a[i]; sb += b[i]; }
    *angular_pairs_host = sa;
    *radial_pairs_host = sa + sb;
    return NEP_OK;
}

int64_t nep_device_bytes(const nep_t* nep)
{
    if (!nep) return 0;
    size_t tot = 0;
    for (int a = 0; a < nep->n_owned; ++a) tot += nep->owned[a].bytes;
    return (int64_t)tot;
}

int nep_probe_fp32(int device, void* cuda_stream, double* tflops_host)
{
    if (!tflops_host) return NEP_ERR_INVALID_ARG;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return NEP_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaGetLastError(); return NEP_ERR_CUDA; }
    float* sink = nullptr;
    if (cudaMalloc((void**)&sink, sizeof(float) * 1024) != cudaSuccess) { cudaGetLastError(); return NEP_ERR_NOMEM; }
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    const int threads = 256, iters = 8192;
    double best = 0.0;
    const int per_sm[4] = {2, 4, 6, 8};                     // resident blocks per SM: the best of the sweep is reported
    for (int sw = 0; sw < 4; ++sw) {
        const int blocks = prop.multiProcessorCount * per_sm[sw];
        for (int rep = 0; rep < 4; ++rep) {
            cudaEventRecord(a, st);
            k_probe_ffma<<<blocks, threads, 0, st>>>(iters, 1e-7f * (float)(rep + 1), sink);
            cudaEventRecord(b, st);
            cudaEventSynchronize(b);
            float ms = 0.0f;
            cudaEventElapsedTime(&ms, a, b);
            const double tf = 2.0 * NEP_PROBE_CHAINS * (double)iters * blocks * threads / (ms * 1e-3) / 1e12;
            if (rep > 0 && tf > best) best = tf;
        }
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(sink);
    if (cudaGetLastError() != cudaSuccess) return NEP_ERR_CUDA;
    *tflops_host = best;
    return NEP_OK;
}

int nep_probe_entry_roundtrip(int device, int32_t count, const int32_t* j_host, const int32_t* slot_host,
                              int32_t* packed_host, int32_t* j_out_host, int32_t* slot_out_host)
{
    if (count < 1 || !j_host || !slot_host || !packed_host || !j_out_host || !slot_out_host) return NEP_ERR_INVALID_ARG;
    for (int32_t a = 0; a < count; ++a)
        if (j_host[a] < 0 || j_host[a] >= NEP_MAX_ATOMS || slot_host[a] < 0 || slot_host[a] >= (1 << NEP_SLOT_BITS)) return NEP_ERR_INVALID_ARG;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return NEP_ERR_CUDA; }
    int32_t* buf = nullptr;
    const size_t bytes = sizeof(int32_t) * (size_t)count;
    if (cudaMalloc((void**)&buf, 5 * bytes) != cudaSuccess) { cudaGetLastError(); return NEP_ERR_NOMEM; }
    cudaMemcpy(buf, j_host, bytes, cudaMemcpyHostToDevice);
    cudaMemcpy(buf + count, slot_host, bytes, cudaMemcpyHostToDevice);
    k_probe_entry<<<div_up(count, 128), 128>>>(count, buf, buf + count, buf + 2 * (size_t)count, buf + 3 * (size_t)count, buf + 4 * (size_t)count);
    cudaMemcpy(packed_host, buf + 2 * (size_t)count, bytes, cudaMemcpyDeviceToHost);
    cudaMemcpy(j_out_host, buf + 3 * (size_t)count, bytes, cudaMemcpyDeviceToHost);
    cudaMemcpy(slot_out_host, buf + 4 * (size_t)count, bytes, cudaMemcpyDeviceToHost);
    cudaFree(buf);
    return cudaGetLastError() == cudaSuccess ? NEP_OK : NEP_ERR_CUDA;
}

}  // extern "C"
