// nep_batch.cuh -- SURVEY.md section 8(f) row 4: population-batched evaluation for training.
//
// SNES evaluates, per generation, a POPULATION of parameter sets on a BATCH of small structures and reduces
// the loss of Eq. (33).  The MD path is built for one large cell; this path is built for
// many small ones:
//   * structures are concatenated (atom_offset[s] .. atom_offset[s+1]); each has its own cell, which may be
//     thinner than 2 r_c: the neighbours of an atom are ALL lattice images within the cutoffs (DESIGN.md reading
//     A18), found once per batch -- the geometry does not depend on the parameters -- by a plain fp64 loop over
//     image shifts, stored per entry as the fp32 pair vector (rounded from the fp64 difference) plus the slot of the
//     reverse entry (j -> i, -N) in j's list;
//   * one launch covers all structures x all members: grid.x runs over the atoms of the batch, grid.y over the
//     members; member p reads its parameters at p * stride from device arrays uploaded once per call (no
//     per-member synchronisation) and stages what a block needs in shared memory;
//   * per member: descriptors (kb_descriptors), network (kb_ann), partial forces of every entry (kb_partial,
//     Eq. (21)), F_i and W_i from the own and the reverse entries (kb_gather, Eqs. (22)-(24));
//   * the data terms of Eq. (33) are reduced on the device per (member, structure) and then per member in a
//     fixed order (kb_loss_partial, kb_loss_total).
// fp32 arithmetic like the MD path, fp64 outputs.  One thread per (atom, member); loops over n, k
// have run-time bounds (any hyper-parameters).  What the kernels take over from the MD path: the entries inside the
// angular cutoff come first in an atom's list (no skipping in place); the radial parts use the per-type basis sums and
// the E^i table (KR operations per pair) in a shared-memory column per thread; the angular coefficients of a pass
// are staged per block as [type pair][k][channel]; five to seven angular channels go in one pass, A_k and B_k are
// formed where they are used; the network has its own kernel with the member's weights in shared memory.
#pragma once
#include "nep_common.cuh"
#include "nep_kernels.cuh"

#define NEP_BATCH_MAX_SHIFT 7      // |image shift relative to the minimum image| per axis that fits the reverse-entry code

struct BatchParams {               // device pointers to the parameters of ALL members, member-major
    const float* cR;               // [n_pop][T][T][NR][KR]
    const float* cA;               // [n_pop][T][T][NA][KA]
    const float* w0;               // [n_pop][H][D]
    const float* b0;               // [n_pop][H]
    const float* w1;               // [n_pop][H]
    const float* b1;               // [n_pop]
};

// ---- neighbour entries with lattice images (reading A18); count pass (fill = 0) and fill pass (fill = 1) --------
__global__ void __launch_bounds__(128)
kb_neighbors(int N, const int* __restrict__ sid, const int* __restrict__ off, const double* __restrict__ Hs,
             const double* __restrict__ Hinvs, const int* __restrict__ Ms, const double* __restrict__ pos,
             const int* __restrict__ type, int n_types, double rcR, float rcA,
             int fill, int cap, int* __restrict__ cnt, int* __restrict__ cntA, int* __restrict__ nbr, float4* __restrict__ dvec,
             unsigned short* __restrict__ code, unsigned char* __restrict__ tnb, int* __restrict__ bad)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    if ((unsigned)type[i] >= (unsigned)n_types) atomicOr(bad, 2);
    const int s = sid[i];
    const double* H = Hs + 9 * s;
    const double* inv = Hinvs + 9 * s;
    const int Ma = Ms[3 * s], Mb = Ms[3 * s + 1], Mc = Ms[3 * s + 2];
    const double rc2 = rcR * rcR;
    const double xi = pos[3 * (size_t)i], yi = pos[3 * (size_t)i + 1], zi = pos[3 * (size_t)i + 2];
    // entries inside the angular cutoff (the fp32 test the kernels apply: r < rcA) are stored first, so that the angular
    // loops of a warp run over the angular entries only instead of skipping the others in place (no divergence)
    int c = 0, ca = 0, cb = fill ? cntA[i] : 0;
    for (int j = off[s]; j < off[s + 1]; ++j) {
        const double tx = __dsub_rn(pos[3 * (size_t)j], xi), ty = __dsub_rn(pos[3 * (size_t)j + 1], yi), tz = __dsub_rn(pos[3 * (size_t)j + 2], zi);
        double n0[3];
#pragma unroll
        for (int k = 0; k < 3; ++k)
            n0[k] = rint(__dadd_rn(__dadd_rn(__dmul_rn(tx, inv[k]), __dmul_rn(ty, inv[3 + k])), __dmul_rn(tz, inv[6 + k])));
        for (int ma = -Ma; ma <= Ma; ++ma)
            for (int mb = -Mb; mb <= Mb; ++mb)
                for (int mc = -Mc; mc <= Mc; ++mc) {
                    const double Na = n0[0] + ma, Nb = n0[1] + mb, Nc = n0[2] + mc;
                    if (j == i && Na == 0.0 && Nb == 0.0 && Nc == 0.0) continue;
                    const double t[3] = {tx, ty, tz};
                    double d[3];
#pragma unroll
                    for (int a = 0; a < 3; ++a)
                        d[a] = __dsub_rn(__dsub_rn(__dsub_rn(t[a], __dmul_rn(Na, H[a])), __dmul_rn(Nb, H[3 + a])), __dmul_rn(Nc, H[6 + a]));
                    const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
                    if (d2 < rc2) {
                        const bool ang = (float)sqrt(d2) < rcA;
                        const int slot = ang ? ca : cb;
                        if (ang) ++ca; else ++cb;
                        if (fill && slot < cap) {
                            const size_t e = (size_t)i * cap + slot;
                            nbr[e] = j;
                            tnb[e] = (unsigned char)type[j];
                            dvec[e] = make_float4((float)d[0], (float)d[1], (float)d[2], (float)sqrt(d2));
                            code[e] = (unsigned short)((ma + 8) | ((mb + 8) << 4) | ((mc + 8) << 8));
                        }
                        ++c;
                    }
                }
    }
    cnt[i] = c;
    if (!fill) cntA[i] = ca;
}

// slot of the reverse entry (j -> i, -N): same atoms, opposite shift relative to the (odd-symmetric) minimum image
__global__ void __launch_bounds__(128)
kb_reverse(int N, int cap, const int* __restrict__ cnt, const int* __restrict__ nbr, const unsigned short* __restrict__ code,
           unsigned short* __restrict__ rev, int* __restrict__ bad)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    for (int m = 0; m < cnt[i]; ++m) {
        const size_t e = (size_t)i * cap + m;
        const int j = nbr[e];
        const unsigned cd = code[e];
        const unsigned want = (16u - (cd & 15u)) | ((16u - ((cd >> 4) & 15u)) << 4) | ((16u - ((cd >> 8) & 15u)) << 8);
        int found = -1;
        for (int mm = 0; mm < cnt[j]; ++mm)
            if (nbr[(size_t)j * cap + mm] == i && code[(size_t)j * cap + mm] == want) { found = mm; break; }
        if (found < 0) { atomicOr(bad, 1); found = 0; }
        rev[e] = (unsigned short)found;
    }
}

// f_k and f_k' of Eqs. (3)-(5) for k = 0..K-1 from the shared basis head:  f_k = (T_k + 1) f_c / 2,
// f_k' = T_k'(x) x'(r) f_c / 2 + (T_k + 1) f_c' / 2
struct ChebWalk {
    BasisHead h; float Tkm1, Tk, Dkm1, Dk; int k;
    __device__ __forceinline__ ChebWalk(float r, float rc_inv) : h(basis_head<true>(r, rc_inv)), Tkm1(1.0f), Tk(1.0f), Dkm1(0.0f), Dk(0.0f), k(0) {}
    __device__ __forceinline__ void get(float& f, float& df) const { f = (Tk + 1.0f) * h.hfc; df = fmaf(Dk, h.hfc_dx, (Tk + 1.0f) * h.hdfc); }
    __device__ __forceinline__ void step()
    {
        if (k == 0) { Tkm1 = 1.0f; Tk = h.x; Dkm1 = 0.0f; Dk = 1.0f; }
        else {
            const float Dn = fmaf(h.two_x, Dk, fmaf(2.0f, Tk, -Dkm1)), Tn = fmaf(h.two_x, Tk, -Tkm1);
            Dkm1 = Dk; Dk = Dn; Tkm1 = Tk; Tk = Tn;
        }
        ++k;
    }
};

// Walk over the entries of one atom (pair vector + distance, neighbour's type), the next entry requested while the
// current one is processed.
struct KbWalk {
    const float4* __restrict__ dv; const unsigned char* __restrict__ tv;
    int m, cnt, t, tn; float4 d, dn;
    __device__ __forceinline__ KbWalk(const float4* __restrict__ dvec_row, const unsigned char* __restrict__ tnb_row, int cnt_)
        : dv(dvec_row), tv(tnb_row), m(-1), cnt(cnt_), t(0), tn(0)
    {
        dn = make_float4(0.0f, 0.0f, 1.0f, 1.0f);
        if (cnt > 0) { dn = dv[0]; tn = tv[0]; }
    }
    __device__ __forceinline__ bool next()
    {
        if (++m >= cnt) return false;
        d = dn; t = tn;
        if (m + 1 < cnt) { dn = dv[m + 1]; tn = tv[m + 1]; }
        return true;
    }
};

// ---- descriptors + network: q, S, Fp, U of one (atom, member) --------------------------------------------------
// scratch per (member, atom): q [D] (also the network input), S [NA][24], fp [D]; row-major, one row per thread
// Shared memory of kb_descriptors / kb_partial (dynamic): this thread's column of T x KR per-type sums (resp. its
// E^i[t][k] table), [t * KR + k][blockDim.x], then the angular coefficients of the current pass, [tp][k][NCHB]
// (zero beyond N_A) -- the member's coefficients are read from global memory once per block, not once per pair.
template <int NCHB>
__device__ __forceinline__ void kb_stage_angular(const NepDims& D, const float* __restrict__ cA, int n0, float* tab)
{
    const int TT = D.T * D.T;
    __syncthreads();                                                     // the previous pass is done with the table
    for (int t = threadIdx.x; t < TT * D.KA * NCHB; t += blockDim.x) {
        const int u = t % NCHB, k = (t / NCHB) % D.KA, tp = t / (NCHB * D.KA);
        tab[t] = (n0 + u < D.NA) ? cA[((size_t)tp * D.NA + n0 + u) * D.KA + k] : 0.0f;
    }
    __syncthreads();
}

template <int NCHB>
__global__ void __launch_bounds__(128)
kb_descriptors(NepDims D, NepCoef C, int N, int cap, BatchParams P, const int* __restrict__ type, const int* __restrict__ cnt,
               const unsigned char* __restrict__ tnb, const float4* __restrict__ dvec,
               float* __restrict__ qbuf, float* __restrict__ Sbuf, const int* __restrict__ cntA)
{
    extern __shared__ float sm[];
    const int BS = blockDim.x, T = D.T;
    float* my = sm + threadIdx.x;
    float* tab = sm + (size_t)T * D.KR * BS;
    const int i0 = blockIdx.x * BS + threadIdx.x;
    const bool valid = i0 < N;
    const int i = valid ? i0 : N - 1;                                    // idle threads shadow the last atom, store nothing
    const int p = blockIdx.y;
    const size_t row = (size_t)p * N + i;
    const int ti = type[i];
    const float* cR = P.cR + (size_t)p * T * T * D.NR * D.KR;
    const float* cA = P.cA + (size_t)p * T * T * D.NA * D.KA;
    float* q = qbuf + row * D.D;
    float* S = Sbuf + row * D.NA * NEP_NUM_S;
    const int c = cnt[i], ca = cntA[i];
    // Eq. (2)-(3) re-associated as in the MD path: q_n = sum_t sum_k c[ti][t][n][k] F_t,k with the per-type basis sums
    // F_t,k = sum_{j of type t} f_k(r_ij): one Chebyshev walk and KR additions per pair, the contraction once per atom
    for (int t = 0; t < T * D.KR; ++t) my[t * BS] = 0.0f;
    for (KbWalk pw(dvec + (size_t)i * cap, tnb + (size_t)i * cap, c); pw.next();) {
        float* F = my + (size_t)pw.t * D.KR * BS;
        ChebWalk w(pw.d.w, D.rcR_inv);
        for (int k = 0; k < D.KR; ++k) {
            float f, df; w.get(f, df);
            F[k * BS] += f;
            w.step();
        }
    }
    for (int n = 0; n < D.NR; ++n) {
        float acc = 0.0f;
        for (int t = 0; t < T; ++t) {
            const float* cc = cR + ((size_t)(ti * T + t) * D.NR + n) * D.KR;
            const float* F = my + (size_t)t * D.KR * BS;
            for (int k = 0; k < D.KR; ++k) acc = fmaf(__ldg(cc + k), F[k * BS], acc);
        }
        if (valid) q[n] = acc;
    }
    // Eq. (12) and Eqs. (13)-(19), NCHB channels at a time (NCHB = N_A for 5..7 channels: one pass)
    for (int n0 = 0; n0 < D.NA; n0 += NCHB) {
        kb_stage_angular<NCHB>(D, cA, n0, tab);
        float Sa[NCHB][NEP_NUM_S];
#pragma unroll
        for (int u = 0; u < NCHB; ++u)
#pragma unroll
            for (int k = 0; k < NEP_NUM_S; ++k) Sa[u][k] = 0.0f;
        for (KbWalk pw(dvec + (size_t)i * cap, tnb + (size_t)i * cap, ca); pw.next();) {
            const float4 d = pw.d;
            const float rinv = 1.0f / d.w;
            const float* cc = tab + (size_t)(ti * T + pw.t) * D.KA * NCHB;
            float g[NCHB];
#pragma unroll
            for (int u = 0; u < NCHB; ++u) g[u] = 0.0f;
            ChebWalk w(d.w, D.rcA_inv);
            for (int k = 0; k < D.KA; ++k) {
                float f, df; w.get(f, df);
#pragma unroll
                for (int u = 0; u < NCHB; ++u) g[u] = fmaf(cc[u], f, g[u]);
                cc += NCHB;
                w.step();
            }
            float b[NEP_NUM_S];
            angular_b(d.x * rinv, d.y * rinv, d.z * rinv, b);
#pragma unroll
            for (int u = 0; u < NCHB; ++u)
#pragma unroll
                for (int k = 0; k < NEP_NUM_S; ++k) Sa[u][k] = fmaf(g[u], b[k], Sa[u][k]);
        }
#pragma unroll
        for (int u = 0; u < NCHB; ++u) {
            const int nn = n0 + u;
            if (nn < D.NA && valid) {
                float out[6];
                q_from_S(Sa[u], C, out);
                for (int l = 0; l < 4; ++l) q[D.NR + l * D.NA + nn] = out[l];
                if (D.has4) q[D.NR + 4 * D.NA + nn] = out[4];
                if (D.has5) q[D.NR + (4 + D.has4) * D.NA + nn] = out[5];
#pragma unroll
                for (int k = 0; k < NEP_NUM_S; ++k) S[nn * NEP_NUM_S + k] = Sa[u][k];
            }
        }
    }
}

// ---- network of one (atom, member): U and Fp = dU/dq, Eq. (1) / Listing 1 -----------------------------------------
// The member's weights are staged once per block in shared memory (rows padded to DP, warp-uniform reads), q sits in
// registers, cf_m = w1_m (1 - tanh^2) in this thread's shared-memory column; as k_ann of the MD path, with the
// per-thread rows of the batch scratch ([row][D]) as input and output.
template <int DP>
__global__ void __launch_bounds__(128)
kb_ann(NepDims D, int N, BatchParams P, const float* __restrict__ qbuf, float* __restrict__ fpbuf, double* __restrict__ energy)
{
    extern __shared__ float sw[];                       // w0 [H][DP], b0 [H], w1 [H], cf [H][128]
    const int p = blockIdx.y;
    const float* w0 = P.w0 + (size_t)p * D.H * D.D;
    for (int t = threadIdx.x; t < D.H * DP; t += 128) { const int m = t / DP, v = t - m * DP; sw[t] = v < D.D ? w0[(size_t)m * D.D + v] : 0.0f; }
    float* sb0 = sw + D.H * DP;
    float* sw1 = sb0 + D.H;
    float* mycf = sw1 + D.H + threadIdx.x;
    for (int t = threadIdx.x; t < D.H; t += 128) { sb0[t] = P.b0[(size_t)p * D.H + t]; sw1[t] = P.w1[(size_t)p * D.H + t]; }
    __syncthreads();
    const int i = blockIdx.x * 128 + threadIdx.x;
    if (i >= N) return;
    const size_t row = (size_t)p * N + i;
    const float* q = qbuf + row * D.D;
    float e = 0.0f;
    {
        float qv[DP];
#pragma unroll
        for (int d = 0; d < DP; ++d) qv[d] = d < D.D ? q[d] : 0.0f;
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
            mycf[m * 128] = w1m * (1.0f - x1 * x1);
        }
    }
    float* fp = fpbuf + row * D.D;
#pragma unroll
    for (int d0 = 0; d0 < DP; d0 += 8) {
        float acc[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) acc[u] = 0.0f;
        const float4* w = reinterpret_cast<const float4*>(sw + d0);
        for (int m = 0; m < D.H; ++m) {
            const float cf = mycf[m * 128];
            const float4 wa = w[m * (DP / 4)], wb = w[m * (DP / 4) + 1];
            acc[0] = fmaf(cf, wa.x, acc[0]); acc[1] = fmaf(cf, wa.y, acc[1]);
            acc[2] = fmaf(cf, wa.z, acc[2]); acc[3] = fmaf(cf, wa.w, acc[3]);
            acc[4] = fmaf(cf, wb.x, acc[4]); acc[5] = fmaf(cf, wb.y, acc[5]);
            acc[6] = fmaf(cf, wb.z, acc[6]); acc[7] = fmaf(cf, wb.w, acc[7]);
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) if (d0 + u < D.D) fp[d0 + u] = acc[u];
    }
    energy[row] = (double)(e - P.b1[p]);
}

// grad P_k(u) of the 24 polynomials on the unit vector (table of SURVEY.md section 8(c)), and the assembly of Eq. (21):
//   pf = [sum_k (B_k - l_k A_k / r) b_k] u + (1/r) sum_k A_k grad P_k(u)
// A_k = sum_n G_nk g_n and B_k = sum_n G_nk g_n' are formed where they are used (no A[24], B[24] in registers).
template <int NCHB>
__device__ __forceinline__ void angular_assemble(const float (&G)[NCHB][NEP_NUM_S], const float* g, const float* dg,
                                                 float x, float y, float z, float rinv, float* pf)
{
    float b[NEP_NUM_S];
    angular_b(x, y, z, b);
    const float x2 = x * x, y2 = y * y, z2 = z * z, xy = x * y, xz = x * z, yz = y * z, xyz = xy * z;
    float cu = 0.0f, vx = 0.0f, vy = 0.0f, vz = 0.0f;
#define KB_USE(k, l, gx, gy, gz)                                                                   \
    { float Ak = G[0][k] * g[0], Bk = G[0][k] * dg[0];                                             \
      _Pragma("unroll") for (int u = 1; u < NCHB; ++u) { Ak = fmaf(G[u][k], g[u], Ak); Bk = fmaf(G[u][k], dg[u], Bk); } \
      cu = fmaf(fmaf(-(float)(l) * rinv, Ak, Bk), b[k], cu); vx = fmaf(Ak, (gx), vx); vy = fmaf(Ak, (gy), vy); vz = fmaf(Ak, (gz), vz); }
    KB_USE(0, 1, 0.0f, 0.0f, 1.0f)
    KB_USE(1, 1, 1.0f, 0.0f, 0.0f)
    KB_USE(2, 1, 0.0f, 1.0f, 0.0f)
    KB_USE(3, 2, -2.0f * x, -2.0f * y, 4.0f * z)
    KB_USE(4, 2, z, 0.0f, x)
    KB_USE(5, 2, 0.0f, z, y)
    KB_USE(6, 2, 2.0f * x, -2.0f * y, 0.0f)
    KB_USE(7, 2, 2.0f * y, 2.0f * x, 0.0f)
    KB_USE(8, 3, -6.0f * xz, -6.0f * yz, -3.0f * (x2 + y2 - 2.0f * z2))
    KB_USE(9, 3, -3.0f * x2 - y2 + 4.0f * z2, -2.0f * xy, 8.0f * xz)
    KB_USE(10, 3, -2.0f * xy, -x2 - 3.0f * y2 + 4.0f * z2, 8.0f * yz)
    KB_USE(11, 3, 2.0f * xz, -2.0f * yz, x2 - y2)
    KB_USE(12, 3, 2.0f * yz, 2.0f * xz, 2.0f * xy)
    KB_USE(13, 3, 3.0f * (x2 - y2), -6.0f * xy, 0.0f)
    KB_USE(14, 3, 6.0f * xy, 3.0f * (x2 - y2), 0.0f)
    KB_USE(15, 4, 12.0f * x * (x2 + y2 - 4.0f * z2), 12.0f * y * (x2 + y2 - 4.0f * z2), -16.0f * z * (3.0f * x2 + 3.0f * y2 - 2.0f * z2))
    KB_USE(16, 4, -z * (9.0f * x2 + 3.0f * y2 - 4.0f * z2), -6.0f * xyz, -3.0f * x * (x2 + y2 - 4.0f * z2))
    KB_USE(17, 4, -6.0f * xyz, -z * (3.0f * x2 + 9.0f * y2 - 4.0f * z2), -3.0f * y * (x2 + y2 - 4.0f * z2))
    KB_USE(18, 4, -4.0f * x * (x2 - 3.0f * z2), 4.0f * y * (y2 - 3.0f * z2), 12.0f * z * (x2 - y2))
    KB_USE(19, 4, -2.0f * y * (3.0f * x2 + y2 - 6.0f * z2), -2.0f * x * (x2 + 3.0f * y2 - 6.0f * z2), 24.0f * xyz)
    KB_USE(20, 4, 3.0f * z * (x2 - y2), -6.0f * xyz, x * (x2 - 3.0f * y2))
    KB_USE(21, 4, 6.0f * xyz, 3.0f * z * (x2 - y2), y * (3.0f * x2 - y2))
    KB_USE(22, 4, 4.0f * x * (x2 - 3.0f * y2), -4.0f * y * (3.0f * x2 - y2), 0.0f)
    KB_USE(23, 4, 4.0f * y * (3.0f * x2 - y2), 4.0f * x * (x2 - 3.0f * y2), 0.0f)
#undef KB_USE
    pf[0] = fmaf(cu, x, rinv * vx); pf[1] = fmaf(cu, y, rinv * vy); pf[2] = fmaf(cu, z, rinv * vz);
}

// ---- partial forces dU_i/dr_ij of every entry, Eq. (21) -----------------------------------------------------------
template <int NCHB>
__global__ void __launch_bounds__(128)
kb_partial(NepDims D, NepCoef C, int N, int cap, BatchParams P, const int* __restrict__ type, const int* __restrict__ cnt,
           const unsigned char* __restrict__ tnb, const float4* __restrict__ dvec, const float* __restrict__ Sbuf,
           const float* __restrict__ fpbuf, float4* __restrict__ pfbuf, const int* __restrict__ cntA)
{
    extern __shared__ float sm[];
    const int BS = blockDim.x, T = D.T;
    float* my = sm + threadIdx.x;
    float* tab = sm + (size_t)T * D.KR * BS;
    const int i0 = blockIdx.x * BS + threadIdx.x;
    const bool valid = i0 < N;
    const int i = valid ? i0 : N - 1;
    const int p = blockIdx.y;
    const size_t row = (size_t)p * N + i;
    const int ti = type[i];
    const float* cR = P.cR + (size_t)p * T * T * D.NR * D.KR;
    const float* cA = P.cA + (size_t)p * T * T * D.NA * D.KA;
    const float* fp = fpbuf + row * D.D;
    const float* S = Sbuf + row * D.NA * NEP_NUM_S;
    float4* pf = pfbuf + row * cap;
    const int c = cnt[i], ca = cntA[i];
    // first term of Eq. (21) re-associated as in the MD path: m_ij = sum_k E^i[tj][k] f_k'(r_ij) with
    // E^i[t][k] = sum_n Fp_n c[ti][t][n][k] formed once per atom (KR FMAs per pair instead of NR x KR)
    for (int t = 0; t < T; ++t)
        for (int k = 0; k < D.KR; ++k) {
            float a = 0.0f;
            for (int n = 0; n < D.NR; ++n) a = fmaf(fp[n], __ldg(cR + ((size_t)(ti * T + t) * D.NR + n) * D.KR + k), a);
            my[(t * D.KR + k) * BS] = a;
        }
    for (KbWalk pw(dvec + (size_t)i * cap, tnb + (size_t)i * cap, c); pw.next();) {
        const int m = pw.m;
        const float4 d = pw.d;
        const float rinv = 1.0f / d.w;
        const float* E = my + (size_t)pw.t * D.KR * BS;
        float s = 0.0f;
        ChebWalk w(d.w, D.rcR_inv);
        for (int k = 0; k < D.KR; ++k) {
            float f, df; w.get(f, df);
            s = fmaf(E[k * BS], df, s);
            w.step();
        }
        if (valid) pf[m] = make_float4(s * d.x * rinv, s * d.y * rinv, s * d.z * rinv, 0.0f);
    }
    // last three terms, NCHB channels at a time (pf is linear in A_k = sum_n G_nk g_n and B_k = sum_n G_nk g_n')
    for (int n0 = 0; n0 < D.NA; n0 += NCHB) {
        kb_stage_angular<NCHB>(D, cA, n0, tab);
        float G[NCHB][NEP_NUM_S];
#pragma unroll
        for (int u = 0; u < NCHB; ++u) {
            const int n = min(n0 + u, D.NA - 1);
            float Sv[NEP_NUM_S], f3[4];
#pragma unroll
            for (int k = 0; k < NEP_NUM_S; ++k) Sv[k] = S[n * NEP_NUM_S + k];
            for (int l = 0; l < 4; ++l) f3[l] = fp[D.NR + l * D.NA + n];
            const float f4 = D.has4 ? fp[D.NR + 4 * D.NA + n] : 0.0f;
            const float f5 = D.has5 ? fp[D.NR + (4 + D.has4) * D.NA + n] : 0.0f;
            G_from_S(Sv, f3, f4, f5, C, G[u]);
            if (n0 + u >= D.NA) {
#pragma unroll
                for (int k = 0; k < NEP_NUM_S; ++k) G[u][k] = 0.0f;
            }
        }
        for (KbWalk pw(dvec + (size_t)i * cap, tnb + (size_t)i * cap, ca); pw.next();) {
            const int m = pw.m;
            const float4 d = pw.d;
            const float rinv = 1.0f / d.w;
            const float* cc = tab + (size_t)(ti * T + pw.t) * D.KA * NCHB;
            float g[NCHB], dg[NCHB];
#pragma unroll
            for (int u = 0; u < NCHB; ++u) { g[u] = 0.0f; dg[u] = 0.0f; }
            ChebWalk w(d.w, D.rcA_inv);
            for (int k = 0; k < D.KA; ++k) {
                float f, df; w.get(f, df);
#pragma unroll
                for (int u = 0; u < NCHB; ++u) { g[u] = fmaf(cc[u], f, g[u]); dg[u] = fmaf(cc[u], df, dg[u]); }
                cc += NCHB;
                w.step();
            }
            float pa[3];
            angular_assemble<NCHB>(G, g, dg, d.x * rinv, d.y * rinv, d.z * rinv, rinv, pa);
            if (valid) {
                float4 o = pf[m];
                o.x += pa[0]; o.y += pa[1]; o.z += pa[2];
                pf[m] = o;
            }
        }
    }
}

// ---- F_i = sum (dU_i/dr_ij - dU_j/dr_ji), W_i = sum r_ij (x) dU_j/dr_ji over all entries (Eqs. 22-24) -----------------
__global__ void __launch_bounds__(128)
kb_gather(int N, int cap, const int* __restrict__ cnt, const int* __restrict__ nbr, const float4* __restrict__ dvec,
          const unsigned short* __restrict__ rev, const float4* __restrict__ pfbuf, double* __restrict__ force, double* __restrict__ virial)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int p = blockIdx.y;
    if (i >= N) return;
    const size_t row = (size_t)p * N + i;
    float f[3] = {0.0f, 0.0f, 0.0f}, w[9];
#pragma unroll
    for (int a = 0; a < 9; ++a) w[a] = 0.0f;
    for (int m = 0; m < cnt[i]; ++m) {
        const size_t e = (size_t)i * cap + m;
        const float4 own = pfbuf[row * cap + m];
        const float4 oth = pfbuf[((size_t)p * N + nbr[e]) * cap + rev[e]];     // dU_j/dr_ji
        const float4 d = dvec[e];
        f[0] += own.x - oth.x; f[1] += own.y - oth.y; f[2] += own.z - oth.z;
        w[0] = fmaf(d.x, oth.x, w[0]); w[1] = fmaf(d.x, oth.y, w[1]); w[2] = fmaf(d.x, oth.z, w[2]);
        w[3] = fmaf(d.y, oth.x, w[3]); w[4] = fmaf(d.y, oth.y, w[4]); w[5] = fmaf(d.y, oth.z, w[5]);
        w[6] = fmaf(d.z, oth.x, w[6]); w[7] = fmaf(d.z, oth.y, w[7]); w[8] = fmaf(d.z, oth.z, w[8]);
    }
    if (force) { force[3 * row] = (double)f[0]; force[3 * row + 1] = (double)f[1]; force[3 * row + 2] = (double)f[2]; }
    if (virial) {
#pragma unroll
        for (int a = 0; a < 9; ++a) virial[9 * row + a] = (double)w[a];
    }
}

// ---- loss of Eq. (33): one block per (structure, member): squared per-structure terms {dU^2, sum |dF|^2, sum dW^2} ----
__global__ void __launch_bounds__(128)
kb_loss_partial(int N, int n_str, const int* __restrict__ off, const double* __restrict__ energy, const double* __restrict__ force,
                const double* __restrict__ virial, const double* __restrict__ u_tar, const double* __restrict__ f_tar,
                const double* __restrict__ w_tar, double* __restrict__ part)
{
    __shared__ double sh[11][128];
    const int s = blockIdx.x, p = blockIdx.y;
    const int a0 = off[s], a1 = off[s + 1];
    double v[11];
#pragma unroll
    for (int a = 0; a < 11; ++a) v[a] = 0.0;
    for (int i = a0 + threadIdx.x; i < a1; i += 128) {          // fixed assignment of atoms to threads: reproducible
        const size_t row = (size_t)p * N + i;
        v[0] += energy[row];
        for (int a = 0; a < 3; ++a) { const double df = force[3 * row + a] - f_tar[3 * (size_t)i + a]; v[1] += df * df; }
        for (int a = 0; a < 9; ++a) v[2 + a] += virial[9 * row + a];
    }
#pragma unroll
    for (int a = 0; a < 11; ++a) sh[a][threadIdx.x] = v[a];
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int a = 0; a < 11; ++a) sh[a][threadIdx.x] += sh[a][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double ns = (double)(a1 - a0);
        const double de = sh[0][0] / ns - u_tar[s];
        const int six[6] = {0, 4, 8, 1, 5, 6};
        double sv = 0.0;
        for (int c = 0; c < 6; ++c) { const double dv = sh[2 + six[c]][0] / ns - w_tar[6 * s + c]; sv += dv * dv; }
        double* o3 = part + 3 * ((size_t)p * n_str + s);
        o3[0] = de * de; o3[1] = sh[1][0]; o3[2] = sv;
    }
}

// one block per member: sums over the structures in a fixed order -> {L_e, L_f, L_v}
__global__ void __launch_bounds__(128)
kb_loss_total(int N, int n_str, const double* __restrict__ part, double* __restrict__ loss)
{
    __shared__ double sh[3][128];
    const int p = blockIdx.x;
    double v[3] = {0.0, 0.0, 0.0};
    for (int s = threadIdx.x; s < n_str; s += 128)
        for (int a = 0; a < 3; ++a) v[a] += part[3 * ((size_t)p * n_str + s) + a];
    for (int a = 0; a < 3; ++a) sh[a][threadIdx.x] = v[a];
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) for (int a = 0; a < 3; ++a) sh[a][threadIdx.x] += sh[a][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        loss[3 * p + 0] = sqrt(sh[0][0] / (double)n_str);
        loss[3 * p + 1] = sqrt(sh[1][0] / (3.0 * (double)N));
        loss[3 * p + 2] = sqrt(sh[2][0] / (6.0 * (double)n_str));
    }
}
