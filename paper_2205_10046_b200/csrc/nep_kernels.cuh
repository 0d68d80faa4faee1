// nep_kernels.cuh -- (a2)-(a8): descriptors, network, partial forces, force/virial accumulation.
//
// One thread per atom in the internal spatial order (adjacent threads = adjacent atoms, so neighbour
// gathers of the 16-byte quantised positions hit L1/L2).  Per-atom arrays are stored [component][atom]
// so that a warp reads/writes 128 contiguous bytes per component.  Kernels per evaluation:
//   k_filter         skin lists -> this step's in-cutoff lists (removes the in-cutoff divergence)
//   k_radial<NR>     Eqs. (2)-(5)      radial descriptor
//   k_angular<NCH>   Eq. (12), (13)-(19) angular sums (24*NCH accumulators in registers) and components
//   k_ann<DP>        Eq. (1) / Listing 1; also E^i[t][k] = sum_n Fp_n c^R[ti][t][n][k]
//   k_force_angular<NCH>  last three terms of Eq. (21): dU_i/dr_ij for every angular pair
//   k_final          first term of Eq. (21) for both directions via the E tables; Eqs. (22)-(24):
//                    scatter-free gather of dU_j/dr_ji through the reverse index
#pragma once
#include "nep_common.cuh"

// Pre-computed coefficients of Eqs. (13)-(19), filled on the host at nep_create.
struct NepCoef {
    float c3[NEP_NUM_S];
    float c4[5];
    float c5[3];
};

// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_filter(NepDims D, const int4* __restrict__ posq, const int4* __restrict__ posq_build,
         const int* __restrict__ listA, const int* __restrict__ cntA,
         const int* __restrict__ listS, const int* __restrict__ cntS,
         int* __restrict__ cA, int* __restrict__ ncA, int* __restrict__ cB, int* __restrict__ ncB,
         unsigned* __restrict__ disp_max)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    {   // displacement since the last list build (reported by nep_max_displacement)
        float dx, dy, dz, r2;
        pair_vec(posq_build[s], pi, D, dx, dy, dz, r2);
        if (r2 > 0.0f) atomicMax(disp_max, __float_as_uint(r2));
    }
    int na = 0, nb = 0;
    const int ca = cntA[s];
    for (int m = 0; m < ca; ++m) {
        const int j = listA[(size_t)m * n + s];
        float dx, dy, dz, r2;
        pair_vec(pi, posq[j], D, dx, dy, dz, r2);
        if (r2 < D.rcA2) { cA[(size_t)na * n + s] = (j << NEP_SLOT_BITS) | m; ++na; }
        else if (r2 < D.rcR2) { cB[(size_t)nb * n + s] = j; ++nb; }
    }
    const int cs = cntS[s];
    for (int m = 0; m < cs; ++m) {
        const int j = listS[(size_t)m * n + s];
        float dx, dy, dz, r2;
        pair_vec(pi, posq[j], D, dx, dy, dz, r2);
        if (r2 < D.rcR2) { cB[(size_t)nb * n + s] = j; ++nb; }
    }
    ncA[s] = na;
    ncB[s] = nb;
}

// ---------------------------------------------------------------------------------------------------
// (a2) q_n = sum_j sum_k c^{ij}_{nk} f_k(r_ij)      Eqs. (2)-(4)
template <int NR>
__global__ void __launch_bounds__(128)
k_radial(NepDims D, const int4* __restrict__ posq, const int* __restrict__ cA, const int* __restrict__ ncA,
         const int* __restrict__ cB, const int* __restrict__ ncB, const float* __restrict__ cR_t,
         float* __restrict__ q)
{
    extern __shared__ float sc[];                       // [T*T][KR][NRP]
    const int tab = D.T * D.T * D.KR * D.NRP;
    for (int t = threadIdx.x; t < tab; t += blockDim.x) sc[t] = cR_t[t];
    __syncthreads();
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    float qn[NR];
#pragma unroll
    for (int a = 0; a < NR; ++a) qn[a] = 0.0f;
    const int na = ncA[s], tot = na + ncB[s];
    for (int m = 0; m < tot; ++m) {
        const int j = (m < na) ? (cA[(size_t)m * n + s] >> NEP_SLOT_BITS) : cB[(size_t)(m - na) * n + s];
        const int4 pj = posq[j];
        float dx, dy, dz, r2;
        pair_vec(pi, pj, D, dx, dy, dz, r2);
        const float r = r2 * rsqrtf(r2);
        const BasisHead h = basis_head<false>(r, D.rcR_inv);
        const float* c = sc + (size_t)((pi.w * D.T + pj.w) * D.KR) * D.NRP;
        float Tkm1 = 1.0f, Tk = h.x;
        float f = 2.0f * h.hfc;                          // k = 0: (T_0 + 1) f_c / 2
#pragma unroll
        for (int a = 0; a < NR; ++a) qn[a] = fmaf(c[a], f, qn[a]);
        if (D.KR > 1) {
            c += D.NRP;
            f = (Tk + 1.0f) * h.hfc;                     // k = 1
#pragma unroll
            for (int a = 0; a < NR; ++a) qn[a] = fmaf(c[a], f, qn[a]);
        }
        for (int k = 2; k < D.KR; ++k) {
            const float Tn = fmaf(h.two_x, Tk, -Tkm1);
            Tkm1 = Tk; Tk = Tn;
            c += D.NRP;
            f = (Tk + 1.0f) * h.hfc;
#pragma unroll
            for (int a = 0; a < NR; ++a) qn[a] = fmaf(c[a], f, qn[a]);
        }
    }
#pragma unroll
    for (int a = 0; a < NR; ++a) q[(size_t)a * n + s] = qn[a];
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

// (a3)+(a4) S_nk = sum_j g_n(r_ij) b_k(r_hat_ij) for n = n0..n0+NCH-1, then the components.
template <int NCH>
__global__ void __launch_bounds__(128)
k_angular(NepDims D, NepCoef C, int n0, const int4* __restrict__ posq, const int* __restrict__ cA,
          const int* __restrict__ ncA, const float* __restrict__ cA_t, float* __restrict__ S_out,
          float* __restrict__ q)
{
    extern __shared__ float sc[];                       // [T*T][KA][NAP]
    const int tab = D.T * D.T * D.KA * D.NAP;
    for (int t = threadIdx.x; t < tab; t += blockDim.x) sc[t] = cA_t[t];
    __syncthreads();
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    float S[NCH][NEP_NUM_S];
#pragma unroll
    for (int a = 0; a < NCH; ++a)
#pragma unroll
        for (int k = 0; k < NEP_NUM_S; ++k) S[a][k] = 0.0f;
    const int na = ncA[s];
    for (int m = 0; m < na; ++m) {
        const int j = cA[(size_t)m * n + s] >> NEP_SLOT_BITS;
        const int4 pj = posq[j];
        float dx, dy, dz, r2;
        pair_vec(pi, pj, D, dx, dy, dz, r2);
        const float rinv = rsqrtf(r2), r = r2 * rinv;
        const BasisHead h = basis_head<false>(r, D.rcA_inv);
        const float* c = sc + (size_t)((pi.w * D.T + pj.w) * D.KA) * D.NAP + n0;
        float g[NCH];
        float Tkm1 = 1.0f, Tk = h.x;
        float f = 2.0f * h.hfc;
#pragma unroll
        for (int a = 0; a < NCH; ++a) g[a] = c[a] * f;
        if (D.KA > 1) {
            c += D.NAP;
            f = (Tk + 1.0f) * h.hfc;
#pragma unroll
            for (int a = 0; a < NCH; ++a) g[a] = fmaf(c[a], f, g[a]);
        }
        for (int k = 2; k < D.KA; ++k) {
            const float Tn = fmaf(h.two_x, Tk, -Tkm1);
            Tkm1 = Tk; Tk = Tn;
            c += D.NAP;
            f = (Tk + 1.0f) * h.hfc;
#pragma unroll
            for (int a = 0; a < NCH; ++a) g[a] = fmaf(c[a], f, g[a]);
        }
        float b[NEP_NUM_S];
        angular_b(dx * rinv, dy * rinv, dz * rinv, b);
#pragma unroll
        for (int a = 0; a < NCH; ++a)
#pragma unroll
            for (int k = 0; k < NEP_NUM_S; ++k) S[a][k] = fmaf(g[a], b[k], S[a][k]);
    }
#pragma unroll
    for (int a = 0; a < NCH; ++a) {
        float out[6];
        q_from_S(S[a], C, out);
        const int nn = n0 + a;
#pragma unroll
        for (int l = 0; l < 4; ++l) q[(size_t)(D.NR + l * D.NA + nn) * n + s] = out[l];
        if (D.has4) q[(size_t)(D.NR + 4 * D.NA + nn) * n + s] = out[4];
        if (D.has5) q[(size_t)(D.NR + (4 + D.has4) * D.NA + nn) * n + s] = out[5];
#pragma unroll
        for (int k = 0; k < NEP_NUM_S; ++k) S_out[(size_t)(nn * NEP_NUM_S + k) * n + s] = S[a][k];
    }
}

// ---------------------------------------------------------------------------------------------------
// (a5) U_i = sum_m w1_m tanh(sum_v w0_mv q_v - b0_m) - b1 and Fp_v = dU_i/dq_v   Eq. (1), Listing 1
// (PAPER.md:52-56, 912-963).  Also the per-atom radial table E^i[t][k] = sum_n Fp_n c^R[ti][t][n][k],
// which turns the radial partial force of Eq. (21) into KR FMAs per pair and direction.
template <int DP>
__global__ void __launch_bounds__(128)
k_ann(NepDims D, const int4* __restrict__ posq, const float* __restrict__ q, const float* __restrict__ w0p,
      const float* __restrict__ b0, const float* __restrict__ w1, float b1, const float* __restrict__ cR_e,
      float* __restrict__ fp, float* __restrict__ U, float* __restrict__ Et)
{
    extern __shared__ float sw[];                       // w0p [H][DP], then b0 [H], w1 [H]
    for (int t = threadIdx.x; t < D.H * DP; t += blockDim.x) sw[t] = w0p[t];
    float* sb0 = sw + D.H * DP;
    float* sw1 = sb0 + D.H;
    for (int t = threadIdx.x; t < D.H; t += blockDim.x) { sb0[t] = b0[t]; sw1[t] = w1[t]; }
    __syncthreads();
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    float qv[DP], fv[DP];
#pragma unroll
    for (int d = 0; d < DP; ++d) { qv[d] = (d < D.D) ? q[(size_t)d * n + s] : 0.0f; fv[d] = 0.0f; }
    float e = 0.0f;
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
        const float cf = w1m * (1.0f - x1 * x1);
#pragma unroll
        for (int d4 = 0; d4 < DP / 4; ++d4) {
            const float4 ww = w[d4];
            fv[4 * d4 + 0] = fmaf(cf, ww.x, fv[4 * d4 + 0]); fv[4 * d4 + 1] = fmaf(cf, ww.y, fv[4 * d4 + 1]);
            fv[4 * d4 + 2] = fmaf(cf, ww.z, fv[4 * d4 + 2]); fv[4 * d4 + 3] = fmaf(cf, ww.w, fv[4 * d4 + 3]);
        }
    }
    U[s] = e - b1;
#pragma unroll
    for (int d = 0; d < DP; ++d) if (d < D.D) fp[(size_t)d * n + s] = fv[d];
    // E table (atom-major so that neighbours can gather a row with 128-bit loads)
    const int ti = posq[s].w;
    for (int t = 0; t < D.T; ++t) {
        const float* c = cR_e + (size_t)((ti * D.T + t) * D.NR) * D.KRP;
        float* out = Et + ((size_t)s * D.T + t) * D.KRP;
        for (int k = 0; k < D.KRP; ++k) {
            float acc = 0.0f;
#pragma unroll
            for (int a = 0; a < 16; ++a) if (a < D.NR && a < DP) acc = fmaf(fv[a < DP ? a : 0], __ldg(c + a * D.KRP + k), acc);
            out[k] = acc;
        }
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
template <int NCH>
__global__ void __launch_bounds__(128)
k_force_angular(NepDims D, NepCoef C, int n0, int accumulate, const int4* __restrict__ posq,
                const int* __restrict__ cA, const int* __restrict__ ncA, const float* __restrict__ cA_t,
                const float* __restrict__ S_in, const float* __restrict__ fp, float4* __restrict__ pf)
{
    extern __shared__ float sc[];                       // [T*T][KA][NAP]
    const int tab = D.T * D.T * D.KA * D.NAP;
    for (int t = threadIdx.x; t < tab; t += blockDim.x) sc[t] = cA_t[t];
    __syncthreads();
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    float G[NCH][NEP_NUM_S];
#pragma unroll
    for (int a = 0; a < NCH; ++a) {
        const int nn = n0 + a;
        float Sv[NEP_NUM_S], f3[4];
#pragma unroll
        for (int k = 0; k < NEP_NUM_S; ++k) Sv[k] = S_in[(size_t)(nn * NEP_NUM_S + k) * n + s];
#pragma unroll
        for (int l = 0; l < 4; ++l) f3[l] = fp[(size_t)(D.NR + l * D.NA + nn) * n + s];
        const float f4 = D.has4 ? fp[(size_t)(D.NR + 4 * D.NA + nn) * n + s] : 0.0f;
        const float f5 = D.has5 ? fp[(size_t)(D.NR + (4 + D.has4) * D.NA + nn) * n + s] : 0.0f;
        G_from_S(Sv, f3, f4, f5, C, G[a]);
    }
    const int na = ncA[s];
    for (int m = 0; m < na; ++m) {
        const int e = cA[(size_t)m * n + s];
        const int j = e >> NEP_SLOT_BITS, slot = e & ((1 << NEP_SLOT_BITS) - 1);
        const int4 pj = posq[j];
        float dx, dy, dz, r2;
        pair_vec(pi, pj, D, dx, dy, dz, r2);
        const float rinv = rsqrtf(r2), r = r2 * rinv;
        const BasisHead h = basis_head<true>(r, D.rcA_inv);
        const float* c = sc + (size_t)((pi.w * D.T + pj.w) * D.KA) * D.NAP + n0;
        float g[NCH], dg[NCH];
        {   // g_n = sum_k c_nk f_k,  g_n' = sum_k c_nk f_k';  f_k' = T_k' (f_c/2) x' + (T_k + 1) f_c'/2
            float Tkm1 = 1.0f, Tk = h.x, Ukm1 = 1.0f, Uk = h.two_x;   // T_0,T_1 ; U_0,U_1
            float f = 2.0f * h.hfc, df = 2.0f * h.hdfc;               // k = 0
#pragma unroll
            for (int a = 0; a < NCH; ++a) { g[a] = c[a] * f; dg[a] = c[a] * df; }
            if (D.KA > 1) {                                          // k = 1: T_1' = U_0 = 1
                c += D.NAP;
                f = (Tk + 1.0f) * h.hfc;
                df = fmaf(Tk + 1.0f, h.hdfc, h.hfc_dx);
#pragma unroll
                for (int a = 0; a < NCH; ++a) { g[a] = fmaf(c[a], f, g[a]); dg[a] = fmaf(c[a], df, dg[a]); }
            }
            for (int k = 2; k < D.KA; ++k) {                         // T_k' = k U_{k-1}
                const float Tn = fmaf(h.two_x, Tk, -Tkm1);
                Tkm1 = Tk; Tk = Tn;
                c += D.NAP;
                f = (Tk + 1.0f) * h.hfc;
                df = fmaf(Tk + 1.0f, h.hdfc, (float)k * Uk * h.hfc_dx);
                const float Un = fmaf(h.two_x, Uk, -Ukm1);
                Ukm1 = Uk; Uk = Un;
#pragma unroll
                for (int a = 0; a < NCH; ++a) { g[a] = fmaf(c[a], f, g[a]); dg[a] = fmaf(c[a], df, dg[a]); }
            }
        }
        const float x = dx * rinv, y = dy * rinv, z = dz * rinv;
        float b[NEP_NUM_S];
        angular_b(x, y, z, b);
        float cu = 0.0f, vx = 0.0f, vy = 0.0f, vz = 0.0f;
        const float x2 = x * x, y2 = y * y, z2 = z * z, xy = x * y, xz = x * z, yz = y * z, xyz = xy * z;
        // ACC(k, l, gradP_k(u)): A_k, B_k, then the two sums
#define NEP_ACC(k, l, gx, gy, gz)                                                                  \
        {                                                                                           \
            float A = 0.0f, B = 0.0f;                                                               \
            _Pragma("unroll") for (int a = 0; a < NCH; ++a) { A = fmaf(G[a][k], g[a], A); B = fmaf(G[a][k], dg[a], B); } \
            cu = fmaf(fmaf(-(float)(l) * rinv, A, B), b[k], cu);                                    \
            vx = fmaf(A, (gx), vx); vy = fmaf(A, (gy), vy); vz = fmaf(A, (gz), vz);                 \
        }
        NEP_ACC(0, 1, 0.0f, 0.0f, 1.0f)
        NEP_ACC(1, 1, 1.0f, 0.0f, 0.0f)
        NEP_ACC(2, 1, 0.0f, 1.0f, 0.0f)
        NEP_ACC(3, 2, -2.0f * x, -2.0f * y, 4.0f * z)
        NEP_ACC(4, 2, z, 0.0f, x)
        NEP_ACC(5, 2, 0.0f, z, y)
        NEP_ACC(6, 2, 2.0f * x, -2.0f * y, 0.0f)
        NEP_ACC(7, 2, 2.0f * y, 2.0f * x, 0.0f)
        NEP_ACC(8, 3, -6.0f * xz, -6.0f * yz, -3.0f * (x2 + y2 - 2.0f * z2))
        NEP_ACC(9, 3, -3.0f * x2 - y2 + 4.0f * z2, -2.0f * xy, 8.0f * xz)
        NEP_ACC(10, 3, -2.0f * xy, -x2 - 3.0f * y2 + 4.0f * z2, 8.0f * yz)
        NEP_ACC(11, 3, 2.0f * xz, -2.0f * yz, x2 - y2)
        NEP_ACC(12, 3, 2.0f * yz, 2.0f * xz, 2.0f * xy)
        NEP_ACC(13, 3, 3.0f * (x2 - y2), -6.0f * xy, 0.0f)
        NEP_ACC(14, 3, 6.0f * xy, 3.0f * (x2 - y2), 0.0f)
        NEP_ACC(15, 4, 12.0f * x * (x2 + y2 - 4.0f * z2), 12.0f * y * (x2 + y2 - 4.0f * z2), -16.0f * z * (3.0f * x2 + 3.0f * y2 - 2.0f * z2))
        NEP_ACC(16, 4, -z * (9.0f * x2 + 3.0f * y2 - 4.0f * z2), -6.0f * xyz, -3.0f * x * (x2 + y2 - 4.0f * z2))
        NEP_ACC(17, 4, -6.0f * xyz, -z * (3.0f * x2 + 9.0f * y2 - 4.0f * z2), -3.0f * y * (x2 + y2 - 4.0f * z2))
        NEP_ACC(18, 4, -4.0f * x * (x2 - 3.0f * z2), 4.0f * y * (y2 - 3.0f * z2), 12.0f * z * (x2 - y2))
        NEP_ACC(19, 4, -2.0f * y * (3.0f * x2 + y2 - 6.0f * z2), -2.0f * x * (x2 + 3.0f * y2 - 6.0f * z2), 24.0f * xyz)
        NEP_ACC(20, 4, 3.0f * z * (x2 - y2), -6.0f * xyz, x * (x2 - 3.0f * y2))
        NEP_ACC(21, 4, 6.0f * xyz, 3.0f * z * (x2 - y2), y * (3.0f * x2 - y2))
        NEP_ACC(22, 4, 4.0f * x * (x2 - 3.0f * y2), -4.0f * y * (3.0f * x2 - y2), 0.0f)
        NEP_ACC(23, 4, 4.0f * y * (3.0f * x2 - y2), 4.0f * x * (x2 - 3.0f * y2), 0.0f)
#undef NEP_ACC
        float4 out = make_float4(fmaf(cu, x, rinv * vx), fmaf(cu, y, rinv * vy), fmaf(cu, z, rinv * vz), 0.0f);
        float4* dst = pf + (size_t)slot * n + s;
        if (accumulate) { const float4 o = *dst; out.x += o.x; out.y += o.y; out.z += o.z; }
        *dst = out;
    }
}

// ---------------------------------------------------------------------------------------------------
// (a6)+(a8) forces and virials.
//  radial: dU_i/dr_ij = [sum_k E^i[tj][k] f_k'(r)] u,  dU_j/dr_ji = -[sum_k E^j[ti][k] f_k'(r)] u
//  angular: dU_i/dr_ij read at own slot, dU_j/dr_ji gathered from j's row at the reverse slot
//  F_i = sum_j (dU_i/dr_ij - dU_j/dr_ji)  (Eqs. 22-23);  W_i = sum_j r_ij (x) dU_j/dr_ji  (Eq. 24)
__global__ void __launch_bounds__(128)
k_final(NepDims D, const int4* __restrict__ posq, const int* __restrict__ perm,
        const int* __restrict__ cA, const int* __restrict__ ncA, const int* __restrict__ cB,
        const int* __restrict__ ncB, const unsigned char* __restrict__ rev, const float* __restrict__ Et,
        const float4* __restrict__ pf, const float* __restrict__ U,
        double* __restrict__ e_out, double* __restrict__ f_out, double* __restrict__ w_out)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= D.n) return;
    const size_t n = (size_t)D.n;
    const int4 pi = posq[s];
    const int ti = pi.w;
    float fx = 0.0f, fy = 0.0f, fz = 0.0f;
    float w[9];
#pragma unroll
    for (int a = 0; a < 9; ++a) w[a] = 0.0f;
    const int na = ncA[s], tot = na + ncB[s];
    const float* Ei = Et + (size_t)s * D.T * D.KRP;
    for (int m = 0; m < tot; ++m) {
        const int j = (m < na) ? (cA[(size_t)m * n + s] >> NEP_SLOT_BITS) : cB[(size_t)(m - na) * n + s];
        const int4 pj = posq[j];
        float dx, dy, dz, r2;
        pair_vec(pi, pj, D, dx, dy, dz, r2);
        const float rinv = rsqrtf(r2), r = r2 * rinv;
        const BasisHead h = basis_head<true>(r, D.rcR_inv);
        const float* ei = Ei + pj.w * D.KRP;
        const float* ej = Et + ((size_t)j * D.T + ti) * D.KRP;
        float Tkm1 = 1.0f, Tk = h.x, Ukm1 = 1.0f, Uk = h.two_x;
        float df = 2.0f * h.hdfc;
        float mi = ei[0] * df, mj = __ldg(ej) * df;
        if (D.KR > 1) {
            df = fmaf(Tk + 1.0f, h.hdfc, h.hfc_dx);
            mi = fmaf(ei[1], df, mi); mj = fmaf(__ldg(ej + 1), df, mj);
        }
        for (int k = 2; k < D.KR; ++k) {
            const float Tn = fmaf(h.two_x, Tk, -Tkm1);
            Tkm1 = Tk; Tk = Tn;
            df = fmaf(Tk + 1.0f, h.hdfc, (float)k * Uk * h.hfc_dx);
            const float Un = fmaf(h.two_x, Uk, -Ukm1);
            Ukm1 = Uk; Uk = Un;
            mi = fmaf(ei[k], df, mi); mj = fmaf(__ldg(ej + k), df, mj);
        }
        const float ux = dx * rinv, uy = dy * rinv, uz = dz * rinv;
        const float ft = mi + mj;                        // (dU_i/dr_ij - dU_j/dr_ji) = (mi + mj) u
        fx = fmaf(ft, ux, fx); fy = fmaf(ft, uy, fy); fz = fmaf(ft, uz, fz);
        const float px = -mj * ux, py = -mj * uy, pz = -mj * uz;   // dU_j/dr_ji
        w[0] = fmaf(dx, px, w[0]); w[1] = fmaf(dx, py, w[1]); w[2] = fmaf(dx, pz, w[2]);
        w[3] = fmaf(dy, px, w[3]); w[4] = fmaf(dy, py, w[4]); w[5] = fmaf(dy, pz, w[5]);
        w[6] = fmaf(dz, px, w[6]); w[7] = fmaf(dz, py, w[7]); w[8] = fmaf(dz, pz, w[8]);
    }
    for (int m = 0; m < na; ++m) {
        const int e = cA[(size_t)m * n + s];
        const int j = e >> NEP_SLOT_BITS, slot = e & ((1 << NEP_SLOT_BITS) - 1);
        const int4 pj = posq[j];
        float dx, dy, dz, r2;
        pair_vec(pi, pj, D, dx, dy, dz, r2);
        const float4 own = pf[(size_t)slot * n + s];
        const int rs = rev[(size_t)slot * n + s];
        const float4 oth = __ldg(pf + (size_t)rs * n + j);
        fx += own.x - oth.x; fy += own.y - oth.y; fz += own.z - oth.z;
        w[0] = fmaf(dx, oth.x, w[0]); w[1] = fmaf(dx, oth.y, w[1]); w[2] = fmaf(dx, oth.z, w[2]);
        w[3] = fmaf(dy, oth.x, w[3]); w[4] = fmaf(dy, oth.y, w[4]); w[5] = fmaf(dy, oth.z, w[5]);
        w[6] = fmaf(dz, oth.x, w[6]); w[7] = fmaf(dz, oth.y, w[7]); w[8] = fmaf(dz, oth.z, w[8]);
    }
    const size_t i = (size_t)perm[s];
    if (e_out) e_out[i] = (double)U[s];
    if (f_out) { f_out[3 * i + 0] = (double)fx; f_out[3 * i + 1] = (double)fy; f_out[3 * i + 2] = (double)fz; }
    if (w_out) {
#pragma unroll
        for (int a = 0; a < 9; ++a) w_out[9 * i + a] = (double)w[a];
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

__global__ void k_kick(int n, double half_dt_conv, const int* __restrict__ type, const double* __restrict__ mass,
                       const double* __restrict__ f, double* __restrict__ vel)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 3 * n) return;
    vel[t] += half_dt_conv * (f[t] / mass[type[t / 3]]);
}
