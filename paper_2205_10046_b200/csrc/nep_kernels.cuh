// nep_kernels.cuh -- (a2)-(a8): descriptors, network, partial forces, force/virial accumulation.
//
// One thread per atom in the internal spatial order (tile-major Morton order of the cells, so that a
// warp's 32 atoms and their neighbours are a compact blob and the neighbour gathers hit L1).  Per-atom
// arrays are stored [component][atom] so that a warp reads/writes 128 contiguous bytes per component.
// Every pair loop is software-pipelined: the entry two pairs ahead and the position one pair ahead
// are in flight while the current pair is computed.  Kernels per evaluation:
//   k_filter              skin lists -> this step's in-cutoff lists + in-cutoff masks (removes the
//                         in-cutoff divergence from every later kernel)
//   k_radial_reg<T,KP> / k_radial_multi<KP,..>   Eqs. (2)-(5) radial descriptor via per-type basis sums
//                         (accumulators in registers for few species, else in shared memory)
//   k_angular<NCH,SM>     Eq. (12), (13)-(19) angular sums (24*NCH accumulators in registers) + components
//   k_ann<DP>             Eq. (1) / Listing 1: U_i and Fp = dU_i/dq
//   k_force_angular<NCH,SM>  last three terms of Eq. (21): dU_i/dr_ij of every angular pair, delivered to j
//   k_force_radial_reg<T,KP> / k_force_radial<KP,..>   first term of Eq. (21): m_ij of every pair, delivered to j
//   k_final               Eqs. (22)-(24): each atom streams what its neighbours delivered (scatter-free on
//                         the read side, no atomics anywhere)
// "Delivered": the sender i stores into row (compact slot of i in j's column) of atom j; that slot is a
// popcount over j's in-cutoff mask below the skin slot of i in j's list (reverse index built with the
// lists), computed inline from a 16-byte gather.
#pragma once
#include "nep_common.cuh"


// Pre-computed coefficients of Eqs. (13)-(19), filled on the host at nep_create.
struct NepCoef {
    float c3[NEP_NUM_S];
    float c4[5];
    float c5[3];
};

// Packed list entry (j << 8) | slot, j < 2^24 = NEP_MAX_ATOMS: all 32 bits are used, so packing and unpacking go
// through unsigned arithmetic (a signed shift would sign-extend every j >= 2^23).
__device__ __forceinline__ int entry_pack(int j, int slot) { return (int)(((unsigned)j << NEP_SLOT_BITS) | (unsigned)slot); }
__device__ __forceinline__ int entry_j(int e) { return (int)((unsigned)e >> NEP_SLOT_BITS); }

// ---------------------------------------------------------------------------------------------------
// Software-pipelined walk over one atom's compact entries  e_m = list[m*n + s] = (j << 8) | rs,
// m = 0..cnt-1: the entry two pairs ahead and the neighbour's position one pair ahead are in flight while
// the current pair is computed.  Usage:
//   PairWalk<MODE> w(...);  while (w.next(D)) { w.j() neighbour, w.pj its posq, w.slot(D) delivery slot }
// MODE 0: positions only.  MODE 1 (cA): also prefetches the neighbour's mask words of the 64-slot group
// of rs, from which slot() = compact slot of this atom in the neighbour's cA column.  MODE 2 (cB): entries
// m < nsplit came from listA, the others from listS (offset by the neighbour's count of outer-shell
// listA entries).  Mask record of an atom (k_filter): 2 W 16-byte pairs, {A_w, O_w} for w < W, then
// {S_w, count}.
// DEPTH = how many pairs ahead the neighbour's position (and mask pair) is requested; the entries run one
// further ahead.
template <int MODE, int DEPTH = 1>
struct PairWalk {
    const int* __restrict__ lp;          // &list[(m + DEPTH + 1) * n + s]
    const int4* __restrict__ posq;
    const ulonglong2* __restrict__ mask;
    size_t n;
    int cnt, m, nsplit;
    int e;               // current entry
    int4 pj;             // current neighbour position
    ulonglong2 mw;       // current neighbour mask pair
    int eq[DEPTH + 1];   // entries m+1 .. m+DEPTH+1
    int4 pq[DEPTH];      // positions of m+1 .. m+DEPTH
    ulonglong2 mq[DEPTH];
    __device__ __forceinline__ PairWalk(const int* __restrict__ list_, size_t n_, int s_, int cnt_,
                                        const int4* __restrict__ posq_, const NepDims& D,
                                        const unsigned long long* __restrict__ mask_ = nullptr, int nsplit_ = 0)
        : lp(list_ + s_), posq(posq_), mask(reinterpret_cast<const ulonglong2*>(mask_)), n(n_), cnt(cnt_), m(-1), nsplit(nsplit_)
    {
#pragma unroll
        for (int d = 0; d <= DEPTH; ++d) { eq[d] = (d < cnt) ? *lp : 0; lp += n; }
#pragma unroll
        for (int d = 0; d < DEPTH; ++d) {
            pq[d] = make_int4(0, 0, 0, 0);
            mq[d] = make_ulonglong2(0ull, 0ull);
            if (d < cnt) fetch(eq[d], d, pq[d], mq[d], D);
        }
    }
    __device__ __forceinline__ void fetch(int ee, int mm, int4& p, ulonglong2& w, const NepDims& D)   // entry ee at position mm
    {
        const int j1 = entry_j(ee);
        p = posq[j1];
        if (MODE >= 1) {
            const int word = (ee & ((1 << NEP_SLOT_BITS) - 1)) >> 6;
            w = mask[(size_t)j1 * (2 * D.maskW) + ((MODE == 2 && mm >= nsplit) ? D.maskW + word : word)];
        }
    }
    __device__ __forceinline__ bool next(const NepDims& D)
    {
        if (++m >= cnt) return false;
        e = eq[0]; pj = pq[0]; mw = mq[0];
#pragma unroll
        for (int d = 0; d < DEPTH; ++d) eq[d] = eq[d + 1];
#pragma unroll
        for (int d = 0; d + 1 < DEPTH; ++d) { pq[d] = pq[d + 1]; mq[d] = mq[d + 1]; }
        if (m + DEPTH < cnt) fetch(eq[DEPTH - 1], m + DEPTH, pq[DEPTH - 1], mq[DEPTH - 1], D);
        if (m + DEPTH + 1 < cnt) eq[DEPTH] = *lp;
        lp += n;
        return true;
    }
    __device__ __forceinline__ int j() const { return entry_j(e); }
    // compact slot of this atom in the neighbour's column of the same list
    __device__ __forceinline__ int slot(const NepDims& D) const
    {
        const int rs = e & ((1 << NEP_SLOT_BITS) - 1);
        const bool fromS = (MODE == 2 && m >= nsplit);
        const unsigned long long word = (MODE == 1 || fromS) ? mw.x : mw.y;
        int cs = __popcll(word & ((1ull << (rs & 63)) - 1ull));
        if (rs >> 6) {                                       // rare: more than 64 skin slots
            const ulonglong2* rec = mask + (size_t)j() * (2 * D.maskW) + (fromS ? D.maskW : 0);
            for (int w = 0; w < (rs >> 6); ++w) cs += __popcll((MODE == 1 || fromS) ? rec[w].x : rec[w].y);
        }
        if (fromS) cs += (int)mw.y;
        return cs;
    }
};

// ---------------------------------------------------------------------------------------------------
// Per-step compaction of the skin lists to this step's in-cutoff lists (removes the in-cutoff divergence
// from every later kernel):
//   cA[m][i] = (j << 8) | rs   pairs with r < rcA,            rs = slot of i in j's SKIN list (rev / revS)
//   cB[m][i] = (j << 8) | rs   pairs with rcA <= r < rcR: first those of listA, then those of listS
// and the mask record of atom i, 2 W 16-byte pairs (W = D.maskW words cover the longest skin list):
//   pair w < W:   .x bit m: slot 64 w + m of listA is inside rcA;  .y: that slot is in the outer shell
//   pair W + w:   .x bit m: slot 64 w + m of listS is inside rcR;  .y: number of outer-shell bits of listA
// The slot of i in j's COMPACT column -- where i delivers dU_i/dr_ij to j -- is the number of set bits
// below rs in the matching mask of j (PairWalk::slot), so no per-step reverse list is built.
template <bool PIPE>
__global__ void __launch_bounds__(256)
k_filter(NepDims D, const int4* __restrict__ posq, const int4* __restrict__ posq_build,
         const int* __restrict__ listA, const int* __restrict__ cntA, const unsigned char* __restrict__ rev,
         const int* __restrict__ listS, const int* __restrict__ cntS, const unsigned char* __restrict__ revS,
         int* __restrict__ cA, int* __restrict__ ncA, int* __restrict__ cB, int* __restrict__ ncB,
         unsigned long long* __restrict__ mask, unsigned* __restrict__ disp_max)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    {   // displacement since the last list build: [0] of this evaluation (nep_max_displacement), [1] the
        // largest of any evaluation since the build (md_step's skin check); one atomic pair per warp
        float dx, dy, dz, r2;
        pair_vec(posq_build[s], pi, D, dx, dy, dz, r2);
        const unsigned am = __activemask();
        const unsigned worst = __reduce_max_sync(am, __float_as_uint(r2));
        if ((threadIdx.x & 31) == (unsigned)(__ffs(am) - 1) && worst > 0u) { atomicMax(disp_max, worst); atomicMax(disp_max + 1, worst); }
    }
    // Branch-free inner loops: the write pointers of the two compact columns advance by n under a predicate,
    // the mask bit of the current slot is shifted along, list / rev pointers step by 4 n per batch.
    ulonglong2* rec = reinterpret_cast<ulonglong2*>(mask) + (size_t)s * (2 * D.maskW);
    int* pa = cA + s;
    int* pb = cB + s;
    int na = 0, nb = 0;
    const size_t n4 = 4 * n;
    {
        // PIPE: the entries of the NEXT batch are requested before the gathers of this one are consumed: a batch then
        // waits for the longer of the two round trips (list column from DRAM, neighbour positions from L1/L2), not for
        // their sum (303 -> 281 us at 1M atoms).  Not beyond ~4M atoms: there the extra rows in flight, each in a page
        // of its own 4 n bytes apart, cost more than they hide (8.19M atoms: 3.52 -> 4.31 ms), and the host picks the
        // plain order, entries of a batch first, then its gathers.
        const int ca = cntA[s];
        const int* lp = listA + s;
        const unsigned char* rp = rev + s;
        int jn[4], rsn[4];
        if (PIPE) {
#pragma unroll
            for (int u = 0; u < 4; ++u) { const bool ok = u < ca; jn[u] = ok ? lp[u * n] : s; rsn[u] = ok ? rp[u * n] : 0; }
            lp += n4; rp += n4;
        }
        for (int w = 0; w < D.maskW; ++w) {
            unsigned long long wa = 0ull, wb = 0ull, bit = 1ull;
            const int mend = min(ca, 64 * (w + 1));
            for (int m0 = 64 * w; m0 < mend; m0 += 4) {          // 4 independent gathers in flight
                int j[4], rs[4]; int4 pj[4];
                if (!PIPE) {
#pragma unroll
                    for (int u = 0; u < 4; ++u) { const bool ok = m0 + u < ca; jn[u] = ok ? lp[u * n] : s; rsn[u] = ok ? rp[u * n] : 0; }
                    lp += n4; rp += n4;
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) { j[u] = jn[u]; rs[u] = rsn[u]; }
#pragma unroll
                for (int u = 0; u < 4; ++u) pj[u] = posq[j[u]];
                if (PIPE) {
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const bool ok = m0 + 4 + u < ca;
                        jn[u] = ok ? lp[u * n] : s;
                        rsn[u] = ok ? rp[u * n] : 0;
                    }
                    lp += n4; rp += n4;
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    float dx, dy, dz, r2;
                    pair_vec(pi, pj[u], D, dx, dy, dz, r2);
                    const int e = entry_pack(j[u], rs[u]);
                    const bool ok = m0 + u < mend;
                    const bool inA = ok && r2 < D.rcA2;
                    const bool inB = ok && !inA && r2 < D.rcR2;
                    if (inA) { *pa = e; pa += n; ++na; wa |= bit; }
                    if (inB) { *pb = e; pb += n; ++nb; wb |= bit; }
                    bit <<= 1;
                }
            }
            rec[w] = make_ulonglong2(wa, wb);
        }
    }
    const unsigned long long nouter = (unsigned long long)nb;
    {
        const int cs = cntS[s];
        const int* lp = listS + s;
        const unsigned char* rp = revS + s;
        int jn[4], rsn[4];
        if (PIPE) {
#pragma unroll
            for (int u = 0; u < 4; ++u) { const bool ok = u < cs; jn[u] = ok ? lp[u * n] : s; rsn[u] = ok ? rp[u * n] : 0; }
            lp += n4; rp += n4;
        }
        for (int w = 0; w < D.maskW; ++w) {
            unsigned long long ws = 0ull, bit = 1ull;
            const int mend = min(cs, 64 * (w + 1));
            for (int m0 = 64 * w; m0 < mend; m0 += 4) {
                int j[4], rs[4]; int4 pj[4];
                if (!PIPE) {
#pragma unroll
                    for (int u = 0; u < 4; ++u) { const bool ok = m0 + u < cs; jn[u] = ok ? lp[u * n] : s; rsn[u] = ok ? rp[u * n] : 0; }
                    lp += n4; rp += n4;
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) { j[u] = jn[u]; rs[u] = rsn[u]; }
#pragma unroll
                for (int u = 0; u < 4; ++u) pj[u] = posq[j[u]];
                if (PIPE) {
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const bool ok = m0 + 4 + u < cs;
                        jn[u] = ok ? lp[u * n] : s;
                        rsn[u] = ok ? rp[u * n] : 0;
                    }
                    lp += n4; rp += n4;
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    float dx, dy, dz, r2;
                    pair_vec(pi, pj[u], D, dx, dy, dz, r2);
                    if (m0 + u < mend && r2 < D.rcR2) { *pb = entry_pack(j[u], rs[u]); pb += n; ++nb; ws |= bit; }
                    bit <<= 1;
                }
            }
            rec[D.maskW + w] = make_ulonglong2(ws, nouter);
        }
    }
    ncA[s] = na;
    ncB[s] = nb;
}

// ---------------------------------------------------------------------------------------------------
// (a2) q_n = sum_j sum_k c^{ij}_{nk} f_k(r_ij)      Eqs. (2)-(4)
// Re-association (exact in real arithmetic): q_n = sum_t sum_k c[ti][t][n][k] F_t,k with the per-type
// basis sums F_t,k = sum_{j of type t} f_k(r_ij), so that a pair costs the Chebyshev recurrence and one
// FMA per k, and the coefficient contraction is done once per atom.  With f_k = (T_k + 1) f_c / 2:
// F_k = A_k + A_0 (k >= 1), F_0 = 2 A_0, where A_k = sum_j T_k(x_ij) f_c(r_ij)/2.

// one pair's contribution to A_0..A_{K-1} held in registers (K compile-time)
template <int KP>
__device__ __forceinline__ void radial_accumulate(float r2, float rc_inv, float* A, int KR = KP)
{
    const float r = r2 * rsqrtf(r2);
    const BasisHead h = basis_head<false>(r, rc_inv);
    A[0] += h.hfc;
    float Tkm1 = 1.0f, Tk = h.x;
    if (KP > 1) A[1] = fmaf(Tk, h.hfc, A[1]);
#pragma unroll
    for (int k = 2; k < KP; ++k) {
        if (k < KP - 3 || k < KR) {                       // uniform: KP - 3 <= KR <= KP
            const float Tn = fmaf(h.two_x, Tk, -Tkm1);
            Tkm1 = Tk; Tk = Tn;
            A[k] = fmaf(Tk, h.hfc, A[k]);
        }
    }
}

// Few species (TT * KP <= 64): the per-type accumulators A[t][k] stay in registers -- no shared memory, so
// the whole L1 serves the neighbour gathers and occupancy is set by registers alone.  The neighbour's
// type selects the row with a 0/1 factor (TT * KR FMAs per pair, no branches).  KP = KR rounded up to 4.
template <int TT, int KP>
__device__ __forceinline__ void radial_accumulate_typed(float r2, float rc_inv, int KR, int tj, float (&A)[TT][KP])
{
    const float r = r2 * rsqrtf(r2);
    const BasisHead h = basis_head<false>(r, rc_inv);
    float v[KP];
    v[0] = h.hfc;
    float Tkm1 = 1.0f, Tk = h.x;
    if (KP > 1) v[1] = Tk * h.hfc;
#pragma unroll
    for (int k = 2; k < KP; ++k) {
        const float Tn = fmaf(h.two_x, Tk, -Tkm1);
        Tkm1 = Tk; Tk = Tn;
        v[k] = Tk * h.hfc;
    }
#pragma unroll
    for (int t = 0; t < TT; ++t) {
        const float sel = (TT == 1 || tj == t) ? 1.0f : 0.0f;
#pragma unroll
        for (int k = 0; k < KP; ++k)
            if (k < KP - 3 || k < KR) A[t][k] = fmaf(sel, v[k], A[t][k]);
    }
}

template <int TT, int KP>
__global__ void __launch_bounds__(128)
k_radial_reg(NepDims D, int tab_stride, const int4* __restrict__ posq, const int* __restrict__ cA,
             const int* __restrict__ ncA, const int* __restrict__ cB, const int* __restrict__ ncB,
             const float* __restrict__ cR_t, float* __restrict__ q)
{
    extern __shared__ float sc[];                        // table [T*T] x tab_stride (rows [k][NRP])
    for (int t = threadIdx.x; t < TT * TT * tab_stride; t += blockDim.x) sc[t] = cR_t[t];
    __syncthreads();
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    float A[TT][KP];
#pragma unroll
    for (int t = 0; t < TT; ++t)
#pragma unroll
        for (int k = 0; k < KP; ++k) A[t][k] = 0.0f;
    {
        PairWalk<0> w(cA, n, s, ncA[s], posq, D);
        while (w.next(D)) {
            float dx, dy, dz, r2;
            pair_vec(pi, w.pj, D, dx, dy, dz, r2);
            radial_accumulate_typed<TT, KP>(r2, D.rcR_inv, D.KR, w.pj.w, A);
        }
    }
    {
        PairWalk<0> w(cB, n, s, ncB[s], posq, D);
        while (w.next(D)) {
            float dx, dy, dz, r2;
            pair_vec(pi, w.pj, D, dx, dy, dz, r2);
            radial_accumulate_typed<TT, KP>(r2, D.rcR_inv, D.KR, w.pj.w, A);
        }
    }
    // F_t,0 = 2 A_t,0 ; F_t,k = A_t,k + A_t,0 ; q_n = sum_t sum_k c[ti][t][n][k] F_t,k
#pragma unroll
    for (int t = 0; t < TT; ++t) {
        const float H = A[t][0];
        A[t][0] = 2.0f * H;
#pragma unroll
        for (int k = 1; k < KP; ++k) A[t][k] += H;
    }
    float* qp = q + s;
    for (int a0 = 0; a0 < D.NR; a0 += 4) {
        float acc[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
        for (int t = 0; t < TT; ++t) {
            const float* c = sc + (size_t)(pi.w * TT + t) * tab_stride + a0;
#pragma unroll
            for (int k = 0; k < KP; ++k) {
                if (k < KP - 3 || k < D.KR) {
#pragma unroll
                    for (int u = 0; u < 4; ++u) acc[u] = fmaf(c[k * D.NRP + u], A[t][k], acc[u]);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) { if (a0 + u < D.NR) *qp = acc[u]; qp += n; }
    }
}

// any number of species: accumulators A[t][k] in shared memory, [t][k][thread] (conflict-free).  KP = KR
// rounded up to a multiple of 4 is a compile-time constant so that the read-modify-write of one pair is
// KR independent LDS, then the recurrence and FMAs, then KR STS; the block size is a compile-time
// constant too, so that every shared-memory offset is an immediate.
template <int KP, int BS>
__device__ __forceinline__ void radial_accumulate_smem(float r2, float rc_inv, int KR, float* acc)
{
    float A[KP];
#pragma unroll
    for (int k = 0; k < KP; ++k) A[k] = (k < KP - 3 || k < KR) ? acc[k * BS] : 0.0f;
    radial_accumulate<KP>(r2, rc_inv, A, KR);
#pragma unroll
    for (int k = 0; k < KP; ++k) if (k < KP - 3 || k < KR) acc[k * BS] = A[k];
}

template <int KP, bool TAB_SM, int BS>
__global__ void __launch_bounds__(BS)
k_radial_multi(NepDims D, int tab_stride, const int4* __restrict__ posq, const int* __restrict__ cA,
               const int* __restrict__ ncA, const int* __restrict__ cB, const int* __restrict__ ncB,
               const float* __restrict__ cR_t, float* __restrict__ q)
{
    extern __shared__ float sm[];                        // A[T][KR][BS], then table [T*T] x tab_stride
    float* sc = sm + (size_t)D.T * D.KR * BS;
    if (TAB_SM) for (int t = threadIdx.x; t < D.T * D.T * tab_stride; t += BS) sc[t] = cR_t[t];
    float* my = sm + threadIdx.x;
    for (int t = 0; t < D.T * D.KR; ++t) my[t * BS] = 0.0f;
    __syncthreads();
    const int s = blockIdx.x * BS + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    const int tstride = D.KR * BS;
    {
        PairWalk<0> w(cA, n, s, ncA[s], posq, D);
        while (w.next(D)) {
            float dx, dy, dz, r2;
            pair_vec(pi, w.pj, D, dx, dy, dz, r2);
            radial_accumulate_smem<KP, BS>(r2, D.rcR_inv, D.KR, my + w.pj.w * tstride);
        }
    }
    {
        PairWalk<0> w(cB, n, s, ncB[s], posq, D);
        while (w.next(D)) {
            float dx, dy, dz, r2;
            pair_vec(pi, w.pj, D, dx, dy, dz, r2);
            radial_accumulate_smem<KP, BS>(r2, D.rcR_inv, D.KR, my + w.pj.w * tstride);
        }
    }
    // q_n = sum_t sum_k c[ti][t][n][k] F_t,k ; table rows [tp][k][NRP], tp stride odd (conflict-free)
    for (int a0 = 0; a0 < D.NR; a0 += 4) {
        float acc[4] = {0.0f, 0.0f, 0.0f, 0.0f};
        for (int t = 0; t < D.T; ++t) {
            const float* A = my + t * tstride;
            const size_t off = (size_t)(pi.w * D.T + t) * tab_stride + a0;
            const float H = A[0];
            float F = 2.0f * H;
            for (int k = 0; k < D.KR; ++k) {
                if (k > 0) F = A[k * BS] + H;
                float c[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) c[u] = TAB_SM ? sc[off + k * D.NRP + u] : __ldg(cR_t + off + k * D.NRP + u);
#pragma unroll
                for (int u = 0; u < 4; ++u) acc[u] = fmaf(c[u], F, acc[u]);
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) if (a0 + u < D.NR) q[(size_t)(a0 + u) * n + s] = acc[u];
    }
}

// ---------------------------------------------------------------------------------------------------
// The 24 angular functions b_k of Eq. (12) on the UNIT vector (x,y,z) (r^2 = 1).
__device__ __forceinline__ void angular_b(float x, float y, float z, float* b)
{
    const float x2 = x * x, y2 = y * y, z2 = z * z;
    const float xy = x * y, xz = x * z, yz = y * z, x2my2 = x2 - y2;
    b[0] = z; b[1] = x; b[2] = y;
    b[3] = 3.0f * z2 - 1.0f; b[4] = xz; b[5] = yz; b[6] = x2my2; b[7] = 2.0f * xy;
    const float f5 = 5.0f * z2 - 1.0f;
    b[8] = (5.0f * z2 - 3.0f) * z; b[9] = f5 * x; b[10] = f5 * y; b[11] = x2my2 * z; b[12] = 2.0f * xy * z;
    b[13] = (x2 - 3.0f * y2) * x; b[14] = (3.0f * x2 - y2) * y;
    const float f7 = 7.0f * z2 - 1.0f, f73 = 7.0f * z2 - 3.0f;
    b[15] = (35.0f * z2 - 30.0f) * z2 + 3.0f; b[16] = f73 * xz; b[17] = f73 * yz;
    b[18] = f7 * x2my2; b[19] = f7 * 2.0f * xy;
    b[20] = (x2 - 3.0f * y2) * xz; b[21] = (3.0f * x2 - y2) * yz;
    b[22] = x2my2 * x2my2 - 4.0f * x2 * y2; b[23] = 4.0f * x2my2 * xy;
}

// Angular components of one n from its 24 sums: out[0..3] = q_n1..q_n4 (Eqs. 13-16), out[4] = q_n222
// (Eq. 18, last line), out[5] = q_n1111 (Eq. 19).
__device__ __forceinline__ void q_from_S(const float* S, const NepCoef& C, float* out)
{
    float a = 0.0f;
#pragma unroll
    for (int k = 0; k < 3; ++k) a = fmaf(C.c3[k] * S[k], S[k], a);
    out[0] = a; a = 0.0f;
#pragma unroll
    for (int k = 3; k < 8; ++k) a = fmaf(C.c3[k] * S[k], S[k], a);
    out[1] = a; a = 0.0f;
#pragma unroll
    for (int k = 8; k < 15; ++k) a = fmaf(C.c3[k] * S[k], S[k], a);
    out[2] = a; a = 0.0f;
#pragma unroll
    for (int k = 15; k < 24; ++k) a = fmaf(C.c3[k] * S[k], S[k], a);
    out[3] = a;
    const float s3 = S[3], s4 = S[4], s5 = S[5], s6 = S[6], s7 = S[7];
    out[4] = C.c4[0] * s3 * s3 * s3 + C.c4[1] * s3 * (s4 * s4 + s5 * s5) + C.c4[2] * s3 * (s6 * s6 + s7 * s7)
           + C.c4[3] * s6 * (s5 * s5 - s4 * s4) + C.c4[4] * s4 * s5 * s7;
    const float s0 = S[0], p = S[1] * S[1] + S[2] * S[2];
    out[5] = C.c5[0] * s0 * s0 * s0 * s0 + C.c5[1] * s0 * s0 * p + C.c5[2] * p * p;
}

// The angular coefficient table of one pass (channels n0 .. n0+NCH-1), per type pair tp = ti*T + tj:
// KAR rows of NCHP = round_up4(NCH) floats.  Row 0 holds csum'_n = 2 c_{n0} + sum_{k>=1} c_{nk}, row k
// (1 <= k < KA) holds c_{nk}, rows KA..KAR-1 are zero (KAR - 1 is a multiple of 4 so that the k loop
// unrolls by 4).  Then   g_n(r) = (f_c/2) [ csum'_n + sum_{k>=1} c_nk T_k(x) ]            (Eqs. 3-4)
// The type-pair stride is an odd number of floats and a row is read with NCH scalar loads: lanes that differ
// in tp hit different banks, lanes with the same tp the same word (broadcast), so every load is one
// wavefront.  (128-bit row loads need fewer instructions but 7 wavefronts per load here -- the 8 lanes of a
// quarter warp share 8 bank groups among up to 25 type pairs -- and this kernel is bound by that pipe.)
// SM = true: the table is staged in shared memory; false: read from global memory (huge tables).
template <bool SM>
__device__ __forceinline__ const float* stage_table(const float* __restrict__ tab_g, int count, float* sc)
{
    if (SM) {
        for (int t = threadIdx.x; t < count; t += blockDim.x) sc[t] = tab_g[t];
        __syncthreads();
        return sc;
    }
    return tab_g;
}

template <int NCH>
__device__ __forceinline__ void load_row(const float* __restrict__ row, float* c)
{
#pragma unroll
    for (int a = 0; a < NCH; ++a) c[a] = row[a];
}

// Warps take 32-atom tiles from a global counter (dynamic, in spatial order): the coefficient table is
// staged once per resident block, and a warp that drew short neighbour lists simply takes the next tile.
__device__ __forceinline__ int next_tile(int* __restrict__ ctr)
{
    int tile = 0;
    if ((threadIdx.x & 31) == 0) tile = atomicAdd(ctr, 1);
    return __shfl_sync(0xffffffffu, tile, 0);
}

// (a3)+(a4) S_nk = sum_j g_n(r_ij) b_k(r_hat_ij) for n = n0..n0+NCH-1, then the components.
template <int NCH>
__device__ __forceinline__ void angular_atom(const NepDims& D, const NepCoef& C, int n0, int tab_stride, const float* tab,
                                             const int4* __restrict__ posq, const int* __restrict__ cA,
                                             const int* __restrict__ ncA, float* __restrict__ S_out,
                                             float* __restrict__ q, int s)
{
    constexpr int N4 = (NCH + 3) / 4;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    // S_nk accumulators as 12 packed pairs per channel: S += g_n * (b_k, b_k+1) is one FFMA2 (sm_100 packed fp32,
    // scalar g broadcast) instead of two FFMA -- the kernel is bound by issue slots, not by the FMA pipe
    float2 S2[NCH][NEP_NUM_S / 2];
#pragma unroll
    for (int a = 0; a < NCH; ++a)
#pragma unroll
        for (int k = 0; k < NEP_NUM_S / 2; ++k) S2[a][k] = make_float2(0.0f, 0.0f);
    const float* tab_i = tab + (size_t)(pi.w * D.T) * tab_stride;
    PairWalk<0> w(cA, n, s, ncA[s], posq, D);
    while (w.next(D)) {
        float dx, dy, dz, r2;
        pair_vec(pi, w.pj, D, dx, dy, dz, r2);
        const float rinv = rsqrtf(r2), r = r2 * rinv;
        const BasisHead h = basis_head<false>(r, D.rcA_inv);
        const float* c4 = tab_i + w.pj.w * tab_stride;
        float g[4 * N4];
        load_row<NCH>(c4, g);                              // csum'
        float Tkm1 = 1.0f, Tk = h.x;
        for (int r0 = 1; r0 < D.KAR; r0 += 4) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                float c[4 * N4];
                load_row<NCH>(c4 + (r0 + u) * (4 * N4), c);
#pragma unroll
                for (int a = 0; a < NCH; ++a) g[a] = fmaf(c[a], Tk, g[a]);
                const float Tn = fmaf(h.two_x, Tk, -Tkm1);
                Tkm1 = Tk; Tk = Tn;
            }
        }
#pragma unroll
        for (int a = 0; a < NCH; ++a) g[a] *= h.hfc;
        float b[NEP_NUM_S];
        angular_b(dx * rinv, dy * rinv, dz * rinv, b);
#pragma unroll
        for (int a = 0; a < NCH; ++a) {
            const float2 ga = make_float2(g[a], g[a]);
#pragma unroll
            for (int k = 0; k < NEP_NUM_S / 2; ++k) S2[a][k] = __ffma2_rn(ga, make_float2(b[2 * k], b[2 * k + 1]), S2[a][k]);
        }
    }
    float* qa = q + (size_t)D.NR * n + s;                  // angular blocks: qa[(blk * NA + nn) * n]
    float* Sp = S_out + (size_t)(n0 * NEP_NUM_S) * n + s;
#pragma unroll
    for (int a = 0; a < NCH; ++a) {
        const int nn = n0 + a;
        if (nn < D.NA) {
            float Sa[NEP_NUM_S];
#pragma unroll
            for (int k = 0; k < NEP_NUM_S / 2; ++k) { Sa[2 * k] = S2[a][k].x; Sa[2 * k + 1] = S2[a][k].y; }
            float out[6];
            q_from_S(Sa, C, out);
            float* qp = qa + (size_t)nn * n;
            const size_t blk = (size_t)D.NA * n;
#pragma unroll
            for (int l = 0; l < 4; ++l) { *qp = out[l]; qp += blk; }
            if (D.has4) { *qp = out[4]; qp += blk; }
            if (D.has5) *qp = out[5];
#pragma unroll
            for (int k = 0; k < NEP_NUM_S; ++k) { *Sp = Sa[k]; Sp += n; }
        }
    }
}

template <int NCH, bool SM>
__global__ void __launch_bounds__(128)
k_angular(NepDims D, NepCoef C, int n0, int tab_stride, const int4* __restrict__ posq, const int* __restrict__ cA,
          const int* __restrict__ ncA, const float* __restrict__ cA_t, float* __restrict__ S_out,
          float* __restrict__ q, int* __restrict__ tile_ctr)
{
    extern __shared__ __align__(16) float sc[];
    const float* tab = stage_table<SM>(cA_t, D.T * D.T * tab_stride, sc);
    const int ntile = (D.n + 31) >> 5;
    for (int tile = next_tile(tile_ctr); tile < ntile; tile = next_tile(tile_ctr)) {
        const int s = tile * 32 + (threadIdx.x & 31);
        if (s < D.n) angular_atom<NCH>(D, C, n0, tab_stride, tab, posq, cA, ncA, S_out, q, s);
    }
}

// ---------------------------------------------------------------------------------------------------
// (a5) U_i = sum_m w1_m tanh(sum_v w0_mv q_v - b0_m) - b1 and Fp_v = dU_i/dq_v   Eq. (1), Listing 1
// (PAPER.md:52-56, 912-963).
template <int DP>
__global__ void __launch_bounds__(128)
k_ann(NepDims D, const float* __restrict__ q, const float* __restrict__ w0p, const float* __restrict__ b0,
      const float* __restrict__ w1, float b1, float* __restrict__ fp, float* __restrict__ U)
{
    // Two phases so that neither holds q and Fp in registers at once (occupancy): forward with q in
    // registers, leaving cf_m = w1_m (1 - tanh^2) in shared memory ([m][thread], conflict-free); backward
    // Fp_v = sum_m cf_m w0_mv eight components at a time.  Weight reads are warp-uniform (broadcast).
    extern __shared__ float sw[];                       // w0p [H][DP], b0 [H], w1 [H], cf [H][BS]
    const int BS = blockDim.x;
    for (int t = threadIdx.x; t < D.H * DP; t += BS) sw[t] = w0p[t];
    float* sb0 = sw + D.H * DP;
    float* sw1 = sb0 + D.H;
    float* scf = sw1 + D.H;
    for (int t = threadIdx.x; t < D.H; t += BS) { sb0[t] = b0[t]; sw1[t] = w1[t]; }
    __syncthreads();
    const int s = blockIdx.x * BS + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    float* mycf = scf + threadIdx.x;
    float e = 0.0f;
    {
        float qv[DP];
#pragma unroll
        for (int d = 0; d < DP; ++d) qv[d] = (d < D.D) ? q[(size_t)d * n + s] : 0.0f;
        for (int m = 0; m < D.H; ++m) {
            const float4* w = reinterpret_cast<const float4*>(sw + m * DP);
            float a0 = -sb0[m], a1 = 0.0f, a2 = 0.0f, a3 = 0.0f;
#pragma unroll
            for (int d4 = 0; d4 < DP / 4; ++d4) {
                const float4 ww = w[d4];
                a0 = fmaf(ww.x, qv[4 * d4 + 0], a0); a1 = fmaf(ww.y, qv[4 * d4 + 1], a1);
                a2 = fmaf(ww.z, qv[4 * d4 + 2], a2); a3 = fmaf(ww.w, qv[4 * d4 + 3], a3);
            }
            const float x1 = tanhf((a0 + a1) + (a2 + a3));
            const float w1m = sw1[m];
            e = fmaf(w1m, x1, e);
            mycf[m * BS] = w1m * (1.0f - x1 * x1);
        }
    }
#pragma unroll
    for (int d0 = 0; d0 < DP; d0 += 8) {
        float acc[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) acc[u] = 0.0f;
        const float4* w = reinterpret_cast<const float4*>(sw + d0);
        for (int m = 0; m < D.H; ++m) {
            const float cf = mycf[m * BS];
            const float4 wa = w[m * (DP / 4)], wb = w[m * (DP / 4) + 1];
            acc[0] = fmaf(cf, wa.x, acc[0]); acc[1] = fmaf(cf, wa.y, acc[1]);
            acc[2] = fmaf(cf, wa.z, acc[2]); acc[3] = fmaf(cf, wa.w, acc[3]);
            acc[4] = fmaf(cf, wb.x, acc[4]); acc[5] = fmaf(cf, wb.y, acc[5]);
            acc[6] = fmaf(cf, wb.z, acc[6]); acc[7] = fmaf(cf, wb.w, acc[7]);
        }
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (d0 + u < D.D) fp[(size_t)(d0 + u) * n + s] = acc[u];
    }
    U[s] = e - b1;
}

// ---------------------------------------------------------------------------------------------------
// (a5) on the tensor cores.  The network is the one dense contraction of the path: z[atoms x H] = q w0^T
// and Fp[atoms x D] = cf w0.  One warp takes a 32-atom tile; mma.sync m16n8k8 TF32 with fp32 accumulation
// and the 3xTF32 split (x = hi + lo, both TF32; acc += lo*hi + hi*lo + hi*hi), which keeps ~fp32 accuracy
// (a plain TF32 product would miss the 1e-5 eV bar by two orders of magnitude).  Weights are split once
// per block into shared memory, in two layouts whose row strides make the B-fragment reads of the forward
// (stride = 12 mod 32) and of the backward pass (stride = 8 mod 32) bank-conflict-free; cf passes through
// a per-warp shared tile (C-fragment layout -> A-fragment layout).  Fragment layouts: PTX ISA, mma.m16n8k8.
// tanh(x) = 1 - 2 / (exp(2x) + 1) with the hardware exp2 and reciprocal (MUFU.EX2, MUFU.RCP): absolute error
// ~1e-7 over the whole range (exact limits +-1), 6 instructions instead of tanhf's ~20; the network's energy bar is
// 1e-5 eV absolute and |w1| < 1.
__device__ __forceinline__ float tanh_fast(float x)
{
    float e;                                               // exp(2x) = 2^(2x log2 e)
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(x * 2.885390081777927f));
    return 1.0f - __fdividef(2.0f, e + 1.0f);
}

__device__ __forceinline__ void tf32_split(float x, unsigned& hi, unsigned& lo)
{
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(hi) : "f"(x));
    const float r = x - __uint_as_float(hi);
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(lo) : "f"(r));
}

__device__ __forceinline__ void mma_tf32(float (&c)[4], const unsigned (&a)[4], unsigned b0, unsigned b1)
{
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

__host__ __device__ __forceinline__ int ann_stride_fwd(int DP) { return DP + ((12 - DP % 32) + 32) % 32; }
__host__ __device__ __forceinline__ int ann_stride_bwd(int DP) { return DP + ((8 - DP % 32) + 32) % 32; }

template <int DP>
__global__ void __launch_bounds__(128)
k_ann_tc(NepDims D, int HP, const float* __restrict__ q, const float* __restrict__ w0p, const float* __restrict__ b0,
         const float* __restrict__ w1, float b1, float* __restrict__ fp, float* __restrict__ U, int* __restrict__ tile_ctr)
{
    constexpr int KT = DP / 8;
    const int SF = ann_stride_fwd(DP), SB = ann_stride_bwd(DP), SC = HP + 4;
    extern __shared__ __align__(16) unsigned smu[];
    unsigned* wfh = smu;                       // [HP][SF] hi, forward layout
    unsigned* wfl = wfh + HP * SF;             // [HP][SF] lo
    unsigned* wbh = wfl + HP * SF;             // [HP][SB] hi, backward layout
    unsigned* wbl = wbh + HP * SB;             // [HP][SB] lo
    float* sb0 = reinterpret_cast<float*>(wbl + HP * SB);   // [HP]
    float* sw1 = sb0 + HP;                                   // [HP]
    float* scf = sw1 + HP + (threadIdx.x >> 5) * 32 * SC;    // this warp's cf tile [32][SC]
    for (int t = threadIdx.x; t < HP * DP; t += blockDim.x) {
        const int m = t / DP, d = t - m * DP;
        unsigned hi, lo;
        tf32_split(m < D.H ? w0p[m * DP + d] : 0.0f, hi, lo);
        wfh[m * SF + d] = hi; wfl[m * SF + d] = lo;
        wbh[m * SB + d] = hi; wbl[m * SB + d] = lo;
    }
    for (int t = threadIdx.x; t < HP; t += blockDim.x) { sb0[t] = t < D.H ? b0[t] : 0.0f; sw1[t] = t < D.H ? w1[t] : 0.0f; }
    __syncthreads();
    const int lane = threadIdx.x & 31, g = lane >> 2, t4 = lane & 3;
    const size_t n = (size_t)D.n;
    const int ntile = (D.n + 31) >> 5, NT = HP >> 3;
    for (int tile = next_tile(tile_ctr); tile < ntile; tile = next_tile(tile_ctr)) {
        const int s0 = tile * 32;
        // A fragments of q (rows = atoms, cols = descriptor components), split once
        unsigned ah[2][KT][4], al[2][KT][4];
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
            for (int kt = 0; kt < KT; ++kt)
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int a = s0 + mt * 16 + g + (r & 1) * 8, d = kt * 8 + t4 + (r >> 1) * 4;
                    const float v = (a < D.n && d < D.D) ? q[(size_t)d * n + a] : 0.0f;
                    tf32_split(v, ah[mt][kt][r], al[mt][kt][r]);
                }
        float e[2][2] = {{0.0f, 0.0f}, {0.0f, 0.0f}};      // [m-tile][row g / g+8] partial energies
        for (int nt = 0; nt < NT; ++nt) {
            float c[2][4];
            {
                const float nb0 = -sb0[nt * 8 + 2 * t4], nb1 = -sb0[nt * 8 + 2 * t4 + 1];
#pragma unroll
                for (int mt = 0; mt < 2; ++mt) { c[mt][0] = nb0; c[mt][1] = nb1; c[mt][2] = nb0; c[mt][3] = nb1; }
            }
            const unsigned* bh = wfh + (nt * 8 + g) * SF + t4;
            const unsigned* bl = wfl + (nt * 8 + g) * SF + t4;
#pragma unroll
            for (int kt = 0; kt < KT; ++kt) {
                const unsigned h0 = bh[kt * 8], h1 = bh[kt * 8 + 4], l0 = bl[kt * 8], l1 = bl[kt * 8 + 4];
#pragma unroll
                for (int mt = 0; mt < 2; ++mt) {
                    mma_tf32(c[mt], al[mt][kt], h0, h1);
                    mma_tf32(c[mt], ah[mt][kt], l0, l1);
                    mma_tf32(c[mt], ah[mt][kt], h0, h1);
                }
            }
            const float w1a = sw1[nt * 8 + 2 * t4], w1b = sw1[nt * 8 + 2 * t4 + 1];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
                const float x0 = tanh_fast(c[mt][0]), x1 = tanh_fast(c[mt][1]), x2 = tanh_fast(c[mt][2]), x3 = tanh_fast(c[mt][3]);
                e[mt][0] = fmaf(w1a, x0, fmaf(w1b, x1, e[mt][0]));
                e[mt][1] = fmaf(w1a, x2, fmaf(w1b, x3, e[mt][1]));
                float* r0 = scf + (mt * 16 + g) * SC + nt * 8 + 2 * t4;
                *reinterpret_cast<float2*>(r0) = make_float2(w1a * (1.0f - x0 * x0), w1b * (1.0f - x1 * x1));
                *reinterpret_cast<float2*>(r0 + 8 * SC) = make_float2(w1a * (1.0f - x2 * x2), w1b * (1.0f - x3 * x3));
            }
        }
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                float v = e[mt][h];
                v += __shfl_xor_sync(0xffffffffu, v, 1);
                v += __shfl_xor_sync(0xffffffffu, v, 2);
                const int a = s0 + mt * 16 + g + h * 8;
                if (t4 == 0 && a < D.n) U[a] = v - b1;
            }
        __syncwarp();
        // backward: Fp[atoms x DP] = cf[atoms x HP] w0[HP x DP]
        float f[2][KT][4];
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
            for (int dt = 0; dt < KT; ++dt)
#pragma unroll
                for (int r = 0; r < 4; ++r) f[mt][dt][r] = 0.0f;
        for (int kt = 0; kt < NT; ++kt) {
            unsigned ch[2][4], cl[2][4];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int r = 0; r < 4; ++r)
                    tf32_split(scf[(mt * 16 + g + (r & 1) * 8) * SC + kt * 8 + t4 + (r >> 1) * 4], ch[mt][r], cl[mt][r]);
            const unsigned* bh = wbh + (kt * 8 + t4) * SB + g;
            const unsigned* bl = wbl + (kt * 8 + t4) * SB + g;
#pragma unroll
            for (int dt = 0; dt < KT; ++dt) {
                const unsigned h0 = bh[dt * 8], h1 = bh[dt * 8 + 4 * SB], l0 = bl[dt * 8], l1 = bl[dt * 8 + 4 * SB];
#pragma unroll
                for (int mt = 0; mt < 2; ++mt) {
                    mma_tf32(f[mt][dt], cl[mt], h0, h1);
                    mma_tf32(f[mt][dt], ch[mt], l0, l1);
                    mma_tf32(f[mt][dt], ch[mt], h0, h1);
                }
            }
        }
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
            for (int dt = 0; dt < KT; ++dt)
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int a = s0 + mt * 16 + g + (r >> 1) * 8, d = dt * 8 + 2 * t4 + (r & 1);
                    if (a < D.n && d < D.D) fp[(size_t)d * n + a] = f[mt][dt][r];
                }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------------
// G_nk = dU_i/dS_nk from Fp and S (chain rule through Eqs. (13)-(19)).
__device__ __forceinline__ void G_from_S(const float* S, const float* f3, float f4, float f5, const NepCoef& C, float* G)
{
#pragma unroll
    for (int k = 0; k < 3; ++k) G[k] = 2.0f * C.c3[k] * S[k] * f3[0];
#pragma unroll
    for (int k = 3; k < 8; ++k) G[k] = 2.0f * C.c3[k] * S[k] * f3[1];
#pragma unroll
    for (int k = 8; k < 15; ++k) G[k] = 2.0f * C.c3[k] * S[k] * f3[2];
#pragma unroll
    for (int k = 15; k < 24; ++k) G[k] = 2.0f * C.c3[k] * S[k] * f3[3];
    const float s3 = S[3], s4 = S[4], s5 = S[5], s6 = S[6], s7 = S[7];
    G[3] += f4 * (3.0f * C.c4[0] * s3 * s3 + C.c4[1] * (s4 * s4 + s5 * s5) + C.c4[2] * (s6 * s6 + s7 * s7));
    G[4] += f4 * (2.0f * C.c4[1] * s3 * s4 - 2.0f * C.c4[3] * s6 * s4 + C.c4[4] * s5 * s7);
    G[5] += f4 * (2.0f * C.c4[1] * s3 * s5 + 2.0f * C.c4[3] * s6 * s5 + C.c4[4] * s4 * s7);
    G[6] += f4 * (2.0f * C.c4[2] * s3 * s6 + C.c4[3] * (s5 * s5 - s4 * s4));
    G[7] += f4 * (2.0f * C.c4[2] * s3 * s7 + C.c4[4] * s4 * s5);
    const float s0 = S[0], s1 = S[1], s2 = S[2], p = s1 * s1 + s2 * s2;
    G[0] += f5 * (4.0f * C.c5[0] * s0 * s0 * s0 + 2.0f * C.c5[1] * s0 * p);
    G[1] += f5 * (2.0f * C.c5[1] * s0 * s0 * s1 + 4.0f * C.c5[2] * p * s1);
    G[2] += f5 * (2.0f * C.c5[1] * s0 * s0 * s2 + 4.0f * C.c5[2] * p * s2);
}

// (a7) dU_i/dr_ij = sum_n sum_k G_nk grad[g_n(r) b_k(r_hat)]            last three terms of Eq. (21)
//   grad[g b_k] = (g' - l_k g / r) b_k(u) u + (g / r) gradP_k(u),  P_k the degree-l_k polynomial of b_k.
// With A_k = sum_n G_nk g_n, B_k = sum_n G_nk g_n':
//   pf = [sum_k (B_k - l_k A_k / r) b_k] u + (1/r) sum_k A_k gradP_k(u).
// g_n and g_n' from the table of k_angular:  with G0_n = sum_{k>=1} c_nk T_k + csum'_n and
// G1_n = sum_{k>=1} c_nk T_k'(x):  g_n = (f_c/2) G0_n,  g_n' = (f_c'/2) G0_n + (f_c/2) x'(r) G1_n;
// T_{k+1}' = 2 T_k + 2 x T_k' - T_{k-1}'.
// NCH channels keep their G_nk in registers; NSM further channels (a pass of 6 or 7) keep them in this thread's
// column of shared memory, [channel * 24 + k][128]: one pass with 48 extra shared loads per pair instead of a
// second pass that would repeat the pair geometry, b_k, grad P_k and the assembly.
template <int NCH, int NSM>
__device__ __forceinline__ void force_angular_atom(const NepDims& D, const NepCoef& C, int n0, int accumulate, int tab_stride,
                                                   const float* tab, const int4* __restrict__ posq,
                                                   const int* __restrict__ cA, const int* __restrict__ ncA,
                                                   const unsigned long long* __restrict__ mask,
                                                   const float* __restrict__ S_in, const float* __restrict__ fp,
                                                   float4* __restrict__ pf, float4* __restrict__ fa, int s,
                                                   float* __restrict__ myG)
{
    constexpr int NT = NCH + NSM;
    constexpr int N4 = (NT + 3) / 4;
    constexpr bool PACKED = NSM > 0;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    float2 G2[NCH][NEP_NUM_S / 2];                          // G_nk in pairs (k, k+1): see NEP_AB
    {
        const float* fpa = fp + (size_t)D.NR * n + s;          // angular blocks: fpa[(blk * NA + nn) * n]
        const size_t blk = (size_t)D.NA * n;
#pragma unroll
        for (int a = 0; a < NT; ++a) {
            const int nn = min(n0 + a, D.NA - 1);
            float Sv[NEP_NUM_S], f3[4];
            const float* Sp = S_in + (size_t)(nn * NEP_NUM_S) * n + s;
#pragma unroll
            for (int k = 0; k < NEP_NUM_S; ++k) { Sv[k] = *Sp; Sp += n; }
            const float* fq = fpa + (size_t)nn * n;
#pragma unroll
            for (int l = 0; l < 4; ++l) { f3[l] = *fq; fq += blk; }
            float f4 = 0.0f, f5 = 0.0f;
            if (D.has4) { f4 = *fq; fq += blk; }
            if (D.has5) f5 = *fq;
            float Gt[NEP_NUM_S];
            G_from_S(Sv, f3, f4, f5, C, Gt);
            if (n0 + a >= D.NA) {                              // padded channel of the global-table fallback
#pragma unroll
                for (int k = 0; k < NEP_NUM_S; ++k) Gt[k] = 0.0f;
            }
#pragma unroll
            for (int k = 0; k < NEP_NUM_S; ++k) {
                if (a < NCH) { if (k & 1) G2[a < NCH ? a : 0][k >> 1].y = Gt[k]; else G2[a < NCH ? a : 0][k >> 1].x = Gt[k]; }
                else myG[((a - NCH) * NEP_NUM_S + k) * 128] = Gt[k];
            }
        }
    }
    const float* tab_i = tab + (size_t)(pi.w * D.T) * tab_stride;
    float sx = 0.0f, sy = 0.0f, sz = 0.0f;                 // sum_j dU_i/dr_ij
    PairWalk<1> w(cA, n, s, ncA[s], posq, D, mask);
    while (w.next(D)) {
        float dx, dy, dz, r2;
        pair_vec(pi, w.pj, D, dx, dy, dz, r2);
        const float rinv = rsqrtf(r2), r = r2 * rinv;
        const BasisHead h = basis_head<true>(r, D.rcA_inv);
        const float* c4 = tab_i + w.pj.w * tab_stride;
        float g[4 * N4], dg[NT];
        load_row<NT>(c4, g);                              // csum'
        {
            // (G0_n, G1_n) += c_nk (T_k, T_k'): one FFMA2 per channel and k (scalar c broadcast)
            float2 gd[NT];
#pragma unroll
            for (int a = 0; a < NT; ++a) gd[a] = make_float2(g[a], 0.0f);
            float Tkm1 = 1.0f, Tk = h.x, Dkm1 = 0.0f, Dk = 1.0f;      // T_0,T_1 ; T_0',T_1'
            for (int r0 = 1; r0 < D.KAR; r0 += 4) {
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    float c[4 * N4];
                    load_row<NT>(c4 + (r0 + u) * (4 * N4), c);
                    const float2 td = make_float2(Tk, Dk);
#pragma unroll
                    for (int a = 0; a < NT; ++a) {
                        if (PACKED) gd[a] = __ffma2_rn(make_float2(c[a], c[a]), td, gd[a]);
                        else { gd[a].x = fmaf(c[a], td.x, gd[a].x); gd[a].y = fmaf(c[a], td.y, gd[a].y); }
                    }
                    const float Dn = fmaf(h.two_x, Dk, fmaf(2.0f, Tk, -Dkm1));
                    const float Tn = fmaf(h.two_x, Tk, -Tkm1);
                    Dkm1 = Dk; Dk = Dn; Tkm1 = Tk; Tk = Tn;
                }
            }
#pragma unroll
            for (int a = 0; a < NT; ++a) {
                const float G0 = gd[a].x;
                g[a] = G0 * h.hfc;
                dg[a] = fmaf(G0, h.hdfc, gd[a].y * h.hfc_dx);
            }
        }
        const float x = dx * rinv, y = dy * rinv, z = dz * rinv;
        float b[NEP_NUM_S];
        angular_b(x, y, z, b);
        float cu = 0.0f, vx = 0.0f, vy = 0.0f, vz = 0.0f;
        const float x2 = x * x, y2 = y * y, z2 = z * z, xy = x * y, xz = x * z, yz = y * z, xyz = xy * z;
        // NEP_AB(kp): (A_k, A_k+1) and (B_k, B_k+1) for k = 2 kp.  PACKED: A += g_n (G_nk, G_nk+1) as one FFMA2 with the
        // scalar g_n broadcast (sm_100 packed fp32).  Measured: with all G in registers (NSM = 0, two warps
        // per scheduler) the packed form is SLOWER (607 -> 645 us at 1M atoms: the kernel waits on dependent chains, not
        // on issue slots); with channels in shared memory (NSM > 0) it is 3 % faster -- hence PACKED = NSM > 0.
        // NEP_USE(k, l, A, B, gradP_k(u)): the two sums.
#define NEP_AB_STEP(kp, a)                                                                         \
            if (PACKED) {                                                                           \
                A2_##kp = __ffma2_rn(make_float2(g[a], g[a]), G2[a][kp], A2_##kp);                  \
                B2_##kp = __ffma2_rn(make_float2(dg[a], dg[a]), G2[a][kp], B2_##kp);                \
            } else {                                                                                \
                A2_##kp.x = fmaf(g[a], G2[a][kp].x, A2_##kp.x); A2_##kp.y = fmaf(g[a], G2[a][kp].y, A2_##kp.y);     \
                B2_##kp.x = fmaf(dg[a], G2[a][kp].x, B2_##kp.x); B2_##kp.y = fmaf(dg[a], G2[a][kp].y, B2_##kp.y);   \
            }
#define NEP_AB(kp)                                                                                 \
        float2 A2_##kp = make_float2(0.0f, 0.0f), B2_##kp = make_float2(0.0f, 0.0f);                \
        _Pragma("unroll") for (int a = 0; a < NCH; ++a) { NEP_AB_STEP(kp, a) }                     \
        _Pragma("unroll") for (int a = 0; a < NSM; ++a) {                                          \
            const float2 Gs = make_float2(myG[(a * NEP_NUM_S + 2 * (kp)) * 128], myG[(a * NEP_NUM_S + 2 * (kp) + 1) * 128]); \
            A2_##kp = __ffma2_rn(make_float2(g[NCH + a], g[NCH + a]), Gs, A2_##kp);                 \
            B2_##kp = __ffma2_rn(make_float2(dg[NCH + a], dg[NCH + a]), Gs, B2_##kp); }
#define NEP_USE(k, l, A, B, gx, gy, gz)                                                            \
        {                                                                                           \
            cu = fmaf(fmaf(-(float)(l) * rinv, (A), (B)), b[k], cu);                                \
            vx = fmaf((A), (gx), vx); vy = fmaf((A), (gy), vy); vz = fmaf((A), (gz), vz);           \
        }
        NEP_AB(0)
        NEP_USE(0, 1, A2_0.x, B2_0.x, 0.0f, 0.0f, 1.0f)
        NEP_USE(1, 1, A2_0.y, B2_0.y, 1.0f, 0.0f, 0.0f)
        NEP_AB(1)
        NEP_USE(2, 1, A2_1.x, B2_1.x, 0.0f, 1.0f, 0.0f)
        NEP_USE(3, 2, A2_1.y, B2_1.y, -2.0f * x, -2.0f * y, 4.0f * z)
        NEP_AB(2)
        NEP_USE(4, 2, A2_2.x, B2_2.x, z, 0.0f, x)
        NEP_USE(5, 2, A2_2.y, B2_2.y, 0.0f, z, y)
        NEP_AB(3)
        NEP_USE(6, 2, A2_3.x, B2_3.x, 2.0f * x, -2.0f * y, 0.0f)
        NEP_USE(7, 2, A2_3.y, B2_3.y, 2.0f * y, 2.0f * x, 0.0f)
        NEP_AB(4)
        NEP_USE(8, 3, A2_4.x, B2_4.x, -6.0f * xz, -6.0f * yz, -3.0f * (x2 + y2 - 2.0f * z2))
        NEP_USE(9, 3, A2_4.y, B2_4.y, -3.0f * x2 - y2 + 4.0f * z2, -2.0f * xy, 8.0f * xz)
        NEP_AB(5)
        NEP_USE(10, 3, A2_5.x, B2_5.x, -2.0f * xy, -x2 - 3.0f * y2 + 4.0f * z2, 8.0f * yz)
        NEP_USE(11, 3, A2_5.y, B2_5.y, 2.0f * xz, -2.0f * yz, x2 - y2)
        NEP_AB(6)
        NEP_USE(12, 3, A2_6.x, B2_6.x, 2.0f * yz, 2.0f * xz, 2.0f * xy)
        NEP_USE(13, 3, A2_6.y, B2_6.y, 3.0f * (x2 - y2), -6.0f * xy, 0.0f)
        NEP_AB(7)
        NEP_USE(14, 3, A2_7.x, B2_7.x, 6.0f * xy, 3.0f * (x2 - y2), 0.0f)
        NEP_USE(15, 4, A2_7.y, B2_7.y, 12.0f * x * (x2 + y2 - 4.0f * z2), 12.0f * y * (x2 + y2 - 4.0f * z2), -16.0f * z * (3.0f * x2 + 3.0f * y2 - 2.0f * z2))
        NEP_AB(8)
        NEP_USE(16, 4, A2_8.x, B2_8.x, -z * (9.0f * x2 + 3.0f * y2 - 4.0f * z2), -6.0f * xyz, -3.0f * x * (x2 + y2 - 4.0f * z2))
        NEP_USE(17, 4, A2_8.y, B2_8.y, -6.0f * xyz, -z * (3.0f * x2 + 9.0f * y2 - 4.0f * z2), -3.0f * y * (x2 + y2 - 4.0f * z2))
        NEP_AB(9)
        NEP_USE(18, 4, A2_9.x, B2_9.x, -4.0f * x * (x2 - 3.0f * z2), 4.0f * y * (y2 - 3.0f * z2), 12.0f * z * (x2 - y2))
        NEP_USE(19, 4, A2_9.y, B2_9.y, -2.0f * y * (3.0f * x2 + y2 - 6.0f * z2), -2.0f * x * (x2 + 3.0f * y2 - 6.0f * z2), 24.0f * xyz)
        NEP_AB(10)
        NEP_USE(20, 4, A2_10.x, B2_10.x, 3.0f * z * (x2 - y2), -6.0f * xyz, x * (x2 - 3.0f * y2))
        NEP_USE(21, 4, A2_10.y, B2_10.y, 6.0f * xyz, 3.0f * z * (x2 - y2), y * (3.0f * x2 - y2))
        NEP_AB(11)
        NEP_USE(22, 4, A2_11.x, B2_11.x, 4.0f * x * (x2 - 3.0f * y2), -4.0f * y * (3.0f * x2 - y2), 0.0f)
        NEP_USE(23, 4, A2_11.y, B2_11.y, 4.0f * y * (3.0f * x2 - y2), 4.0f * x * (x2 - 3.0f * y2), 0.0f)
#undef NEP_AB
#undef NEP_AB_STEP
#undef NEP_USE
        float4 out = make_float4(fmaf(cu, x, rinv * vx), fmaf(cu, y, rinv * vy), fmaf(cu, z, rinv * vz), 0.0f);
        sx += out.x; sy += out.y; sz += out.z;
        // delivered to the receiver: row (slot of i in j's column) of atom j -- a fire-and-forget store
        // here instead of a dependent gather in k_final; only this thread ever touches that element
        float4* dst = pf + (size_t)w.slot(D) * n + w.j();
        if (accumulate) { const float4 o = *dst; out.x += o.x; out.y += o.y; out.z += o.z; }
        *dst = out;
    }
    if (accumulate) { const float4 o = fa[s]; sx += o.x; sy += o.y; sz += o.z; }
    fa[s] = make_float4(sx, sy, sz, 0.0f);
}

template <int NCH, int NSM, bool SM>
__global__ void __launch_bounds__(128)
k_force_angular(NepDims D, NepCoef C, int n0, int accumulate, int tab_stride, const int4* __restrict__ posq,
                const int* __restrict__ cA, const int* __restrict__ ncA, const unsigned long long* __restrict__ mask,
                const float* __restrict__ cA_t, const float* __restrict__ S_in, const float* __restrict__ fp,
                float4* __restrict__ pf, float4* __restrict__ fa, int* __restrict__ tile_ctr)
{
    extern __shared__ __align__(16) float sc[];         // [coefficient table (SM)] [G of the NSM channels: NSM * 24 rows of 128]
    const float* tab = stage_table<SM>(cA_t, D.T * D.T * tab_stride, sc);
    float* myG = sc + (SM ? D.T * D.T * tab_stride : 0) + threadIdx.x;
    const int ntile = (D.n + 31) >> 5;
    for (int tile = next_tile(tile_ctr); tile < ntile; tile = next_tile(tile_ctr)) {
        const int s = tile * 32 + (threadIdx.x & 31);
        if (s < D.n) force_angular_atom<NCH, NSM>(D, C, n0, accumulate, tab_stride, tab, posq, cA, ncA, mask, S_in, fp, pf, fa, s, myG);
    }
}

// ---------------------------------------------------------------------------------------------------
// (a6) radial partial forces, sender side.   dU_i/dr_ij = m_ij u_ij  (first term of Eq. (21)) with
//   m_ij = sum_k E^i[tj][k] f_k'(r_ij),   E^i[t][k] = sum_n Fp_n c^R[ti][t][n][k]
// (an exact re-association of sum_n Fp_n g_n'(r_ij): KR FMAs per pair instead of NR x KR).
//   f_k' = P_k + f_c'/2 with P_k = T_k f_c'/2 + T_k' (f_c/2) x':  P_0 = f_c'/2, P_1 = x f_c'/2 + (f_c/2) x',
//   P_{k+1} = 2 x P_k - P_{k-1} + 2 (f_c/2) x' T_k   (from T_{k+1}' = 2 T_k + 2 x T_k' - T_{k-1}')
// The scalar m_ij is delivered to the receiver j (a fire-and-forget store; only this thread ever touches
// that element): mA[slot][j] for the angular-range pairs, mB[slot][j] for the outer shell.  (Not into the
// .w of pf: a 4-byte write into a sector that has left L2 costs a DRAM read-modify-write.)  The own sum  sum_j m_ij u_ij  is added to fa[i].
// E^i lives in shared memory, [t][k][thread] (conflict-free), T x KR rows: as little as possible, because
// shared memory is carved out of the L1 that serves the neighbour gathers.
template <int KP, int BS>
__device__ __forceinline__ float radial_m(float r, float rc_inv, int KR, const float* __restrict__ E)
{
    const BasisHead h = basis_head<true>(r, rc_inv);
    const float c2 = 2.0f * h.hfc_dx;
    float Ta = 1.0f, Tb = h.x, Pa = h.hdfc, Pb = fmaf(h.x, h.hdfc, h.hfc_dx);
    float Ev[KP];
#pragma unroll
    for (int k = 0; k < KP; ++k) Ev[k] = (k < KP - 3 || k < KR) ? E[k * BS] : 0.0f;
    float m0 = 0.0f, m1 = 0.0f;
#pragma unroll
    for (int k = 0; k < KP; ++k) {
        if (k < KP - 3 || k < KR) {                   // uniform: KP - 3 <= KR <= KP
            const float df = Pa + h.hdfc;             // f_k'
            if (k & 1) m1 = fmaf(Ev[k], df, m1); else m0 = fmaf(Ev[k], df, m0);
            const float Pn = fmaf(h.two_x, Pb, fmaf(c2, Tb, -Pa));
            const float Tn = fmaf(h.two_x, Tb, -Ta);
            Pa = Pb; Pb = Pn; Ta = Tb; Tb = Tn;
        }
    }
    return m0 + m1;
}

// register variant for few species (TT * KP <= 64): E^i[t][k] in registers, all TT dot products per pair,
// the neighbour's type selects one -- no shared memory beyond the staged coefficient table.
template <int TT, int KP>
__device__ __forceinline__ float radial_m_typed(float r, float rc_inv, int KR, int tj, const float (&E)[TT][KP])
{
    const BasisHead h = basis_head<true>(r, rc_inv);
    const float c2 = 2.0f * h.hfc_dx;
    float Ta = 1.0f, Tb = h.x, Pa = h.hdfc, Pb = fmaf(h.x, h.hdfc, h.hfc_dx);
    float m[TT];
#pragma unroll
    for (int t = 0; t < TT; ++t) m[t] = 0.0f;
#pragma unroll
    for (int k = 0; k < KP; ++k) {
        if (k < KP - 3 || k < KR) {                   // uniform: KP - 3 <= KR <= KP
            const float df = Pa + h.hdfc;             // f_k'
#pragma unroll
            for (int t = 0; t < TT; ++t) m[t] = fmaf(E[t][k], df, m[t]);
            const float Pn = fmaf(h.two_x, Pb, fmaf(c2, Tb, -Pa));
            const float Tn = fmaf(h.two_x, Tb, -Ta);
            Pa = Pb; Pb = Pn; Ta = Tb; Tb = Tn;
        }
    }
    float out = m[0];
#pragma unroll
    for (int t = 1; t < TT; ++t) out = (tj == t) ? m[t] : out;
    return out;
}

template <int TT, int KP>
__global__ void __launch_bounds__(128)
k_force_radial_reg(NepDims D, const int4* __restrict__ posq, const int* __restrict__ cA, const int* __restrict__ ncA,
                   const int* __restrict__ cB, const int* __restrict__ ncB, const unsigned long long* __restrict__ mask,
                   const float* __restrict__ fp, const float* __restrict__ cR_e, float* __restrict__ mA,
                   float* __restrict__ mB, float4* __restrict__ fa)
{
    extern __shared__ __align__(16) float sc[];          // cR_e [T*T][NR][KP]
    {
        const int cnt4 = TT * TT * D.NR * (KP / 4);
        for (int t = threadIdx.x; t < cnt4; t += blockDim.x) reinterpret_cast<float4*>(sc)[t] = reinterpret_cast<const float4*>(cR_e)[t];
        __syncthreads();
    }
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    float E[TT][KP];
    {
#pragma unroll
        for (int t = 0; t < TT; ++t)
#pragma unroll
            for (int k = 0; k < KP; ++k) E[t][k] = 0.0f;
        const float* fpa = fp + s;
        for (int a = 0; a < D.NR; ++a) {
            const float f = *fpa;
            fpa += n;
#pragma unroll
            for (int t = 0; t < TT; ++t) {
                const float4* c = reinterpret_cast<const float4*>(sc) + (size_t)((pi.w * TT + t) * D.NR + a) * (KP / 4);
#pragma unroll
                for (int k4 = 0; k4 < KP / 4; ++k4) {
                    const float4 cc = c[k4];
                    E[t][4 * k4 + 0] = fmaf(f, cc.x, E[t][4 * k4 + 0]); E[t][4 * k4 + 1] = fmaf(f, cc.y, E[t][4 * k4 + 1]);
                    E[t][4 * k4 + 2] = fmaf(f, cc.z, E[t][4 * k4 + 2]); E[t][4 * k4 + 3] = fmaf(f, cc.w, E[t][4 * k4 + 3]);
                }
            }
        }
    }
    float fx = 0.0f, fy = 0.0f, fz = 0.0f;
    {
        PairWalk<1> w(cA, n, s, ncA[s], posq, D, mask);
        while (w.next(D)) {
            float dx, dy, dz, r2;
            pair_vec(pi, w.pj, D, dx, dy, dz, r2);
            const float rinv = rsqrtf(r2);
            const float m = radial_m_typed<TT, KP>(r2 * rinv, D.rcR_inv, D.KR, w.pj.w, E);
            const float mr = m * rinv;
            fx = fmaf(mr, dx, fx); fy = fmaf(mr, dy, fy); fz = fmaf(mr, dz, fz);
            mA[(size_t)w.slot(D) * n + w.j()] = m;
        }
    }
    {
        const int nsplit = (int)mask[(size_t)s * D.mrec + 2 * D.maskW + 1];
        PairWalk<2> w(cB, n, s, ncB[s], posq, D, mask, nsplit);
        while (w.next(D)) {
            float dx, dy, dz, r2;
            pair_vec(pi, w.pj, D, dx, dy, dz, r2);
            const float rinv = rsqrtf(r2);
            const float m = radial_m_typed<TT, KP>(r2 * rinv, D.rcR_inv, D.KR, w.pj.w, E);
            const float mr = m * rinv;
            fx = fmaf(mr, dx, fx); fy = fmaf(mr, dy, fy); fz = fmaf(mr, dz, fz);
            mB[(size_t)w.slot(D) * n + w.j()] = m;
        }
    }
    float4 own = fa[s];
    own.x += fx; own.y += fy; own.z += fz;
    fa[s] = own;
}

template <int KP, bool TAB_SM, int BS>
__global__ void __launch_bounds__(BS)
k_force_radial(NepDims D, const int4* __restrict__ posq, const int* __restrict__ cA, const int* __restrict__ ncA,
               const int* __restrict__ cB, const int* __restrict__ ncB, const unsigned long long* __restrict__ mask,
               const float* __restrict__ fp, const float* __restrict__ cR_e, float* __restrict__ mA,
               float* __restrict__ mB, float4* __restrict__ fa)
{
    extern __shared__ __align__(16) float sm[];          // E [T][KR][BS] (16-byte padded), then cR_e [T*T][NR][KP]
    float* sc = sm + (size_t)round_up4_dev(D.T * D.KR) * BS;
    if (TAB_SM) {
        const int cnt4 = D.T * D.T * D.NR * (KP / 4);
        for (int t = threadIdx.x; t < cnt4; t += BS) reinterpret_cast<float4*>(sc)[t] = reinterpret_cast<const float4*>(cR_e)[t];
        __syncthreads();
    }
    const int s = blockIdx.x * BS + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    float* my = sm + threadIdx.x;
    {   // E^i[t][k] from the radial components of Fp (re-read per neighbour type: L1 hits)
        const float4* tab4 = reinterpret_cast<const float4*>(TAB_SM ? sc : cR_e);
        for (int t = 0; t < D.T; ++t) {
            const float4* c = tab4 + (size_t)((pi.w * D.T + t) * D.NR) * (KP / 4);
            float4 acc[KP / 4];
#pragma unroll
            for (int k4 = 0; k4 < KP / 4; ++k4) acc[k4] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            const float* fpa = fp + s;
            for (int a = 0; a < D.NR; ++a) {
                const float f = *fpa;
                fpa += n;
#pragma unroll
                for (int k4 = 0; k4 < KP / 4; ++k4) {
                    const float4 cc = TAB_SM ? c[a * (KP / 4) + k4] : __ldg(c + a * (KP / 4) + k4);
                    acc[k4].x = fmaf(f, cc.x, acc[k4].x); acc[k4].y = fmaf(f, cc.y, acc[k4].y);
                    acc[k4].z = fmaf(f, cc.z, acc[k4].z); acc[k4].w = fmaf(f, cc.w, acc[k4].w);
                }
            }
            float* e = my + (size_t)(t * D.KR) * BS;
#pragma unroll
            for (int k4 = 0; k4 < KP / 4; ++k4) {
                const float v[4] = {acc[k4].x, acc[k4].y, acc[k4].z, acc[k4].w};
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (4 * k4 + u < KP - 3 || 4 * k4 + u < D.KR) e[(4 * k4 + u) * BS] = v[u];
            }
        }
    }
    const int tstride = D.KR * BS;
    float fx = 0.0f, fy = 0.0f, fz = 0.0f;
    {
        PairWalk<1> w(cA, n, s, ncA[s], posq, D, mask);
        while (w.next(D)) {
            float dx, dy, dz, r2;
            pair_vec(pi, w.pj, D, dx, dy, dz, r2);
            const float rinv = rsqrtf(r2);
            const float m = radial_m<KP, BS>(r2 * rinv, D.rcR_inv, D.KR, my + w.pj.w * tstride);
            const float mr = m * rinv;
            fx = fmaf(mr, dx, fx); fy = fmaf(mr, dy, fy); fz = fmaf(mr, dz, fz);
            mA[(size_t)w.slot(D) * n + w.j()] = m;
        }
    }
    {
        const int nsplit = (int)mask[(size_t)s * D.mrec + 2 * D.maskW + 1];
        PairWalk<2> w(cB, n, s, ncB[s], posq, D, mask, nsplit);
        while (w.next(D)) {
            float dx, dy, dz, r2;
            pair_vec(pi, w.pj, D, dx, dy, dz, r2);
            const float rinv = rsqrtf(r2);
            const float m = radial_m<KP, BS>(r2 * rinv, D.rcR_inv, D.KR, my + w.pj.w * tstride);
            const float mr = m * rinv;
            fx = fmaf(mr, dx, fx); fy = fmaf(mr, dy, fy); fz = fmaf(mr, dz, fz);
            mB[(size_t)w.slot(D) * n + w.j()] = m;
        }
    }
    float4 own = fa[s];
    own.x += fx; own.y += fy; own.z += fz;
    fa[s] = own;
}

// ---------------------------------------------------------------------------------------------------
// (a8) forces and virials, receiver side.  Row m of this atom's columns holds what neighbour j = cA[m][i]
// (or cB[m][i]) delivered: dU_j/dr_ji = pf[m][i].xyz - mA[m][i] u_ij  (angular part, radial scalar m_ji;
// u_ji = -u_ij), resp. -mB[m][i] u_ij for the outer shell -- coalesced reads, no gather of partial
// forces, no atomics.  fa[i] = sum_j dU_i/dr_ij (both parts).
//   F_i = sum_j (dU_i/dr_ij - dU_j/dr_ji)  (Eqs. 22-23);  W_i = sum_j r_ij (x) dU_j/dr_ji  (Eq. 24)
struct FinalAcc {
    float fx, fy, fz, w[9];
};

__device__ __forceinline__ void final_pair(FinalAcc& acc, float dx, float dy, float dz, float px, float py, float pz)
{
    acc.fx -= px; acc.fy -= py; acc.fz -= pz;
    acc.w[0] = fmaf(dx, px, acc.w[0]); acc.w[1] = fmaf(dx, py, acc.w[1]); acc.w[2] = fmaf(dx, pz, acc.w[2]);
    acc.w[3] = fmaf(dy, px, acc.w[3]); acc.w[4] = fmaf(dy, py, acc.w[4]); acc.w[5] = fmaf(dy, pz, acc.w[5]);
    acc.w[6] = fmaf(dz, px, acc.w[6]); acc.w[7] = fmaf(dz, py, acc.w[7]); acc.w[8] = fmaf(dz, pz, acc.w[8]);
}

// one list of one atom, four pairs at a time: the four entries of the next batch, then the four neighbour
// positions and the four received records of this batch are in flight together (the kernel is bound by
// memory latency, not arithmetic)
template <bool ANG>
__device__ __forceinline__ void final_walk(const NepDims& D, const int4& pi, const int4* __restrict__ posq,
                                           const int* __restrict__ lp, const float* __restrict__ colm,
                                           const float4* __restrict__ colp, int cnt, FinalAcc& acc)
{
    const size_t n = (size_t)D.n;
    int en[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) en[u] = (u < cnt) ? lp[(size_t)u * n] : 0;
    for (int m0 = 0; m0 < cnt; m0 += 4) {
        int4 pj[4]; float mv[4]; float4 pv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) pj[u] = posq[entry_j(en[u])];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (m0 + u < cnt) {
                mv[u] = colm[(size_t)(m0 + u) * n];
                if (ANG) pv[u] = colp[(size_t)(m0 + u) * n];
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) en[u] = (m0 + 4 + u < cnt) ? lp[(size_t)(m0 + 4 + u) * n] : 0;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (m0 + u < cnt) {
                float dx, dy, dz, r2;
                pair_vec(pi, pj[u], D, dx, dy, dz, r2);
                const float rinv = rsqrtf(r2);
                const float sr = -mv[u] * rinv;
                if (ANG) final_pair(acc, dx, dy, dz, fmaf(sr, dx, pv[u].x), fmaf(sr, dy, pv[u].y), fmaf(sr, dz, pv[u].z));
                else final_pair(acc, dx, dy, dz, sr * dx, sr * dy, sr * dz);
            }
        }
    }
}

__global__ void __launch_bounds__(256)
k_final(NepDims D, const int4* __restrict__ posq, const int* __restrict__ perm,
        const int* __restrict__ cA, const int* __restrict__ ncA, const int* __restrict__ cB,
        const int* __restrict__ ncB, const float4* __restrict__ pf, const float* __restrict__ mA, const float* __restrict__ mB,
        const float4* __restrict__ fa, const float* __restrict__ U,
        double* __restrict__ e_out, double* __restrict__ f_out, double* __restrict__ w_out)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= D.n) return;
    const int4 pi = posq[s];
    FinalAcc acc;
    {
        const float4 own = fa[s];
        acc.fx = own.x; acc.fy = own.y; acc.fz = own.z;
    }
#pragma unroll
    for (int a = 0; a < 9; ++a) acc.w[a] = 0.0f;
    final_walk<true>(D, pi, posq, cA + s, mA + s, pf + s, ncA[s], acc);
    final_walk<false>(D, pi, posq, cB + s, mB + s, nullptr, ncB[s], acc);
    const size_t i = (size_t)perm[s];
    if (e_out) e_out[i] = (double)U[s];
    if (f_out) { f_out[3 * i + 0] = (double)acc.fx; f_out[3 * i + 1] = (double)acc.fy; f_out[3 * i + 2] = (double)acc.fz; }
    if (w_out) {
#pragma unroll
        for (int a = 0; a < 9; ++a) w_out[9 * i + a] = (double)acc.w[a];
    }
}

// ---------------------------------------------------------------------------------------------------
// test hooks: [component][atom] sorted -> [atom][component] caller's order
__global__ void k_export_rows(int n, int ncomp, const int* __restrict__ perm, const float* __restrict__ in,
                              float* __restrict__ out)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const size_t i = (size_t)perm[s];
    for (int c = 0; c < ncomp; ++c) out[i * ncomp + c] = in[(size_t)c * n + s];
}

// ---------------------------------------------------------------------------------------------------
// latent-space vector of every atom,
//   latent[i][mu] = w1_mu tanh(sum_v w0_mu,v q_v - b0_mu)      (hidden-layer state of Eq. (1) times w1)
// from the descriptors of the last evaluation; output [n][H] fp32 in the caller's atom order.  One thread
// per atom with q in registers, weights staged in shared memory (warp-uniform reads), as in k_ann.
template <int DP>
__global__ void __launch_bounds__(128)
k_latent(NepDims D, const int* __restrict__ perm, const float* __restrict__ q, const float* __restrict__ w0p,
         const float* __restrict__ b0, const float* __restrict__ w1, float* __restrict__ out)
{
    extern __shared__ float sw[];                       // w0p [H][DP], b0 [H], w1 [H]
    for (int t = threadIdx.x; t < D.H * DP; t += blockDim.x) sw[t] = w0p[t];
    float* sb0 = sw + D.H * DP;
    float* sw1 = sb0 + D.H;
    for (int t = threadIdx.x; t < D.H; t += blockDim.x) { sb0[t] = b0[t]; sw1[t] = w1[t]; }
    __syncthreads();
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    float qv[DP];
#pragma unroll
    for (int d = 0; d < DP; ++d) qv[d] = (d < D.D) ? q[(size_t)d * n + s] : 0.0f;
    float* row = out + (size_t)perm[s] * D.H;
    for (int m = 0; m < D.H; ++m) {
        const float4* w = reinterpret_cast<const float4*>(sw + m * DP);
        float a0 = -sb0[m], a1 = 0.0f, a2 = 0.0f, a3 = 0.0f;
#pragma unroll
        for (int d4 = 0; d4 < DP / 4; ++d4) {
            const float4 ww = w[d4];
            a0 = fmaf(ww.x, qv[4 * d4 + 0], a0); a1 = fmaf(ww.y, qv[4 * d4 + 1], a1);
            a2 = fmaf(ww.z, qv[4 * d4 + 2], a2); a3 = fmaf(ww.w, qv[4 * d4 + 3], a3);
        }
        row[m] = sw1[m] * tanhf((a0 + a1) + (a2 + a3));
    }
}

// ---------------------------------------------------------------------------------------------------
// per-atom heat current J_i = W_i . v_i, Eq. (25), and the total J = sum_i J_i,
// Eq. (26), from the per-atom virial of the last evaluation (W[3a+b], caller's order,
// fp64) and the caller's velocities: J_i^a = sum_b W_i^{ab} v_i^b.  The total is reduced in a fixed
// order (block partials, then one block), so it is reproducible run to run.
__global__ void __launch_bounds__(256)
k_heat_current(int n, const double* __restrict__ w, const double* __restrict__ vel, double* __restrict__ j_atom,
               double* __restrict__ partial)
{
    __shared__ double sh[3][256];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double j[3] = {0.0, 0.0, 0.0};
    if (i < n) {
        const double* W = w + 9 * (size_t)i;
        const double vx = vel[3 * (size_t)i + 0], vy = vel[3 * (size_t)i + 1], vz = vel[3 * (size_t)i + 2];
#pragma unroll
        for (int a = 0; a < 3; ++a) j[a] = W[3 * a + 0] * vx + W[3 * a + 1] * vy + W[3 * a + 2] * vz;
        if (j_atom) { j_atom[3 * (size_t)i + 0] = j[0]; j_atom[3 * (size_t)i + 1] = j[1]; j_atom[3 * (size_t)i + 2] = j[2]; }
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) sh[a][threadIdx.x] = j[a];
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int a = 0; a < 3; ++a) sh[a][threadIdx.x] += sh[a][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x < 3) partial[3 * (size_t)blockIdx.x + threadIdx.x] = sh[threadIdx.x][0];
}

__global__ void __launch_bounds__(256)
k_heat_total(int nblocks, const double* __restrict__ partial, double* __restrict__ j_total)
{
    __shared__ double sh[3][256];
    double j[3] = {0.0, 0.0, 0.0};
    for (int b = threadIdx.x; b < nblocks; b += 256) {     // fixed assignment of partials to threads
#pragma unroll
        for (int a = 0; a < 3; ++a) j[a] += partial[3 * (size_t)b + a];
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) sh[a][threadIdx.x] = j[a];
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int a = 0; a < 3; ++a) sh[a][threadIdx.x] += sh[a][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x < 3) j_total[threadIdx.x] = sh[threadIdx.x][0];
}

// ---------------------------------------------------------------------------------------------------
// (a9) velocity-Verlet pieces, caller's atom order, fp64 state.
__global__ void k_kick_drift(int n, double half_dt_conv, double dt, const int* __restrict__ type,
                             const double* __restrict__ mass, const double* __restrict__ f,
                             double* __restrict__ vel, double* __restrict__ pos)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 3 * n) return;
    const double a = f[t] / mass[type[t / 3]];
    const double v = vel[t] + half_dt_conv * a;
    vel[t] = v;
    pos[t] += dt * v;
}

// second half kick of one step fused with the first half kick + drift of the next (NVE, same forces): the
// two kicks are applied one after the other, exactly as the separate kernels would
__global__ void k_kick_kick_drift(int n, double half_dt_conv, double dt, const int* __restrict__ type,
                                  const double* __restrict__ mass, const double* __restrict__ f,
                                  double* __restrict__ vel, double* __restrict__ pos)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 3 * n) return;
    const double a = f[t] / mass[type[t / 3]];
    double v = vel[t] + half_dt_conv * a;
    v = v + half_dt_conv * a;
    vel[t] = v;
    pos[t] += dt * v;
}

__global__ void k_kick(int n, double half_dt_conv, const int* __restrict__ type, const double* __restrict__ mass,
                       const double* __restrict__ f, double* __restrict__ vel)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 3 * n) return;
    vel[t] += half_dt_conv * (f[t] / mass[type[t / 3]]);
}

// ---------------------------------------------------------------------------------------------------
// Berendsen thermostat (reading A15), applied after the second half
// kick: sum_i m_i v_i^2 by block partials and one final block (fixed order: reproducible), then
// v *= lambda, lambda = sqrt(1 + (dt/tau) (T_target / T - 1)), T = sum m v^2 / (conv 3 N k_B); all on the
// device, no host round trip.
__global__ void __launch_bounds__(256)
k_mv2_partial(int n, const int* __restrict__ type, const double* __restrict__ mass, const double* __restrict__ vel,
              double* __restrict__ partial)
{
    __shared__ double sh[256];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double a = 0.0;
    if (i < n) {
        const double vx = vel[3 * (size_t)i + 0], vy = vel[3 * (size_t)i + 1], vz = vel[3 * (size_t)i + 2];
        a = mass[type[i]] * (vx * vx + vy * vy + vz * vz);
    }
    sh[threadIdx.x] = a;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

// one block: total of the partials -> scale factor lambda in out[0], temperature before the rescale in out[1]
__global__ void __launch_bounds__(256)
k_berendsen_lambda(int nblocks, const double* __restrict__ partial, double inv_conv_3nkb, double dt_over_tau,
                   double t_target, double* __restrict__ out)
{
    __shared__ double sh[256];
    double a = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += 256) a += partial[b];
    sh[threadIdx.x] = a;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double T = sh[0] * inv_conv_3nkb;
        out[0] = T > 0.0 ? sqrt(fmax(0.0, 1.0 + dt_over_tau * (t_target / T - 1.0))) : 1.0;
        out[1] = T;
    }
}

// Langevin thermostat half step (reading A16): v <- c1 v + c2 sqrt(k_B T / m) R per component,
// R a counter-based standard normal deviate: SplitMix64 finaliser of seed + (2 c + h) * 0x9E3779B97F4A7C15,
// h = 0, 1 -> u = ((x >> 11) + 1/2) 2^-53 -> Box-Muller; counter c = (draw * n + i) * 3 + a.
__device__ __forceinline__ unsigned long long splitmix_mix(unsigned long long z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

__device__ __forceinline__ double counter_normal(unsigned long long seed, unsigned long long c)
{
    const unsigned long long x0 = splitmix_mix(seed + (2ull * c) * 0x9E3779B97F4A7C15ull);
    const unsigned long long x1 = splitmix_mix(seed + (2ull * c + 1ull) * 0x9E3779B97F4A7C15ull);
    const double u0 = ((double)(x0 >> 11) + 0.5) * (1.0 / 9007199254740992.0);
    const double u1 = ((double)(x1 >> 11) + 0.5) * (1.0 / 9007199254740992.0);
    return sqrt(-2.0 * log(u0)) * cos(2.0 * 3.14159265358979323846 * u1);
}

__global__ void k_langevin_half(int n, double c1, double c2, double kt_conv, unsigned long long seed, unsigned long long draw,
                                const int* __restrict__ type, const double* __restrict__ mass, double* __restrict__ vel)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 3 * n) return;
    const int i = t / 3;
    const double sig = sqrt(kt_conv / mass[type[i]]);             // sqrt(k_B T conv / m), Angstrom / fs
    vel[t] = c1 * vel[t] + c2 * sig * counter_normal(seed, draw * (unsigned long long)n * 3ull + (unsigned long long)t);
}

__global__ void k_scale_velocities(int n3, const double* __restrict__ lambda, double* __restrict__ vel)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n3) vel[t] *= lambda[0];
}

// ---------------------------------------------------------------------------------------------------
// Data terms of the loss, Eq. (33) (reading A17), of the last evaluation: block
// partials of {sum U_i, sum |F_i - F_i^tar|^2, sum W_i[0..8]} (11 numbers), then one block adds them in a
// fixed order.
__global__ void __launch_bounds__(256)
k_loss_partial(int n, const double* __restrict__ e, const double* __restrict__ f, const double* __restrict__ w,
               const double* __restrict__ f_target, double* __restrict__ partial)
{
    __shared__ double sh[11][256];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double v[11];
#pragma unroll
    for (int a = 0; a < 11; ++a) v[a] = 0.0;
    if (i < n) {
        v[0] = e[i];
#pragma unroll
        for (int a = 0; a < 3; ++a) { const double d = f[3 * (size_t)i + a] - f_target[3 * (size_t)i + a]; v[1] += d * d; }
#pragma unroll
        for (int a = 0; a < 9; ++a) v[2 + a] = w[9 * (size_t)i + a];
    }
#pragma unroll
    for (int a = 0; a < 11; ++a) sh[a][threadIdx.x] = v[a];
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int a = 0; a < 11; ++a) sh[a][threadIdx.x] += sh[a][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x < 11) partial[11 * (size_t)blockIdx.x + threadIdx.x] = sh[threadIdx.x][0];
}

__global__ void __launch_bounds__(256)
k_loss_total(int nblocks, const double* __restrict__ partial, double* __restrict__ total)
{
    __shared__ double sh[11][256];
    double v[11];
#pragma unroll
    for (int a = 0; a < 11; ++a) v[a] = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += 256) {
#pragma unroll
        for (int a = 0; a < 11; ++a) v[a] += partial[11 * (size_t)b + a];
    }
#pragma unroll
    for (int a = 0; a < 11; ++a) sh[a][threadIdx.x] = v[a];
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int a = 0; a < 11; ++a) sh[a][threadIdx.x] += sh[a][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x < 11) total[threadIdx.x] = sh[threadIdx.x][0];
}
