// nep_common.cuh -- context, device-side constants and small device helpers shared by the kernels
// of the B200-native NEP3 library.  (Product code: shares nothing with oracle/.)
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/nep.h"

#define NEP_MAX_TYPES 16
#define NEP_NUM_S 24            // sums S_{n,k}, k = 0..23 (Eq. 12)
#define NEP_NCH_MAX 7           // most angular n-values handled per pass (24*NCH accumulators in registers)
#define NEP_SLOT_BITS 8         // packed angular entry: (j << 8) | skin slot
#define NEP_MAX_ATOMS (1 << 24)

// Kernel ids for the optional per-kernel CUDA-event timing (nep_profile_*; bench.py's roofline leg).
enum NepKernelId {
    NEP_K_CELL_HIST = 0, NEP_K_SCAN, NEP_K_SCATTER, NEP_K_SORT_CELLS, NEP_K_QUANTIZE, NEP_K_BUILD_LISTS,
    NEP_K_BUILD_REV, NEP_K_FILTER, NEP_K_RADIAL, NEP_K_ANGULAR, NEP_K_ANN, NEP_K_FORCE_ANGULAR, NEP_K_FORCE_RADIAL, NEP_K_FINAL,
    NEP_K_KICK_DRIFT, NEP_K_KICK, NEP_K_THERMOSTAT, NEP_K_EXPORT, NEP_K_BATCH, NEP_K_BATCH_DESC, NEP_K_BATCH_ANN, NEP_K_BATCH_PARTIAL,
    NEP_K_BATCH_GATHER, NEP_K_BATCH_LOSS, NEP_K_COUNT
};
#define NEP_PROF_PAIRS 32768     // event pairs kept before a forced drain

// ---------------------------------------------------------------------------------------------------
// Scalars every kernel needs; passed by value as a kernel argument (lives in the constant bank).
struct NepDims {
    int n;                       // atoms
    int T, NR, KR, NA, KA, D, H;
    int NRP, NAP;                // NR, NA rounded up to a multiple of 4 (row stride of the c tables)
    int KRP;                     // KR rounded up to 4 (row stride of the per-atom E table)
    int KAR;                     // rows of an angular coefficient table: 1 + (KA - 1 rounded up to 4)
    int nblk, has4, has5;        // descriptor blocks after the radial one; 4-/5-body present
    float rcR, rcA, rcR_inv, rcA_inv, rcR2, rcA2;
    float h[9];                  // cell rows a, b, c times 2^-32: quantised fractional units -> Angstrom
    int tri;                     // the cell has off-diagonal elements (general 3x3 product in pair_vec)
    int capA, capS;              // storage rows of the skin lists (angular-range part, outer shell)
    int maskW;                   // 64-bit words of one in-cutoff mask (covers the longest skin list)
    int mrec;                    // 64-bit words of an atom's mask record (4 maskW, see k_filter)
};

struct nep_ctx {
    nep_hyper_t h;
    NepDims d;
    int device;
    cudaStream_t stream;
    char err[512];
    int64_t launches;

    // per-kernel timing (off by default): one event pair per launch on `stream`, drained on read
    bool prof_on;
    cudaEvent_t* prof_ev;    // [2 * NEP_PROF_PAIRS], created on first enable
    int* prof_kid;           // [NEP_PROF_PAIRS] kernel id of each pair
    int prof_used;
    double prof_ms[NEP_K_COUNT];
    int64_t prof_n[NEP_K_COUNT];

    // model (device)
    float* cR_t;     // [T*T] x strideR: rows [k][NRP]   c_radial with the n-values of one k contiguous
    float* cA_t;     // per angular pass: [T*T] x pass_stride: KAR rows of round_up4(nch) floats (see k_angular)
    int n_pass;              // angular passes (channels n0 .. n0+nch-1 each)
    int pass_n0[16], pass_nch[16], pass_off[16], pass_stride[16];   // offsets / strides in floats
    bool angular_tab_smem;   // tables staged in shared memory (else read from global memory)
    int* tile_ctr;           // [64] device: dynamic tile counters of the angular kernels (zeroed per evaluation)
    int num_sms;
    float* cR_e;     // [T(ti)][T(tj)][NR][KRP]  for the per-atom E table of k_force_radial
    int strideR;            // odd type-pair stride (floats) of cR_t: bank-conflict-free lookups
    int KP;                 // KR rounded up to a multiple of 4
    int nch_max;            // angular n-values per pass (<= NEP_NCH_MAX)
    size_t smem_budget;     // shared memory per SM that the table-in-smem kernels may carve out of L1
    bool ann_fp32;          // NEP_ANN_FP32 set: the fp32-FMA network kernel instead of the tensor-core one
    bool ann_precise;       // sum_m |w1_m| too large for tanh_fast's absolute error (upload_parameters): k_ann with tanhf
    double raggedness;      // of the last build: sum over warps of 32 x longest list / sum of list lengths
    bool force_smem_radial; // NEP_RADIAL_SMEM set: use the shared-memory radial kernels even where a register variant exists
    float* w0p;      // [H][DP] rows padded with zeros to DP
    float* b0;       // [H]
    float* w1;       // [H]
    float b1;
    int DP;          // descriptor length padded to the ANN kernel's tier
    double mass[NEP_MAX_TYPES];
    double* mass_dev;

    // system
    int64_t n;
    double H[9], Hinv[9];    // cell rows a, b, c (Angstrom) and the inverse (fractional s = r Hinv)
    double volume;
    double skin;
    int ncell[3];
    int ntile[3];            // 4-cell tiles per axis
    int64_t n_cells;         // padded: ntile[0]*ntile[1]*ntile[2]*64
    bool have_lists;
    bool have_eval;          // internal E/F/W hold an evaluation
    bool force_current;      // ... and it belongs to the positions md_step will continue from
    const double* force_pos_tag;
    int steps_since_build;
    int maxA_skin, maxR_skin, maxS_skin;   // list sizes of the last build (angular-range part; radial = A + shell; shell)

    // per-atom (device); "sorted" = internal spatial order, "orig" = caller's order
    int* type_orig;          // [n]
    int* perm;               // [n] sorted -> orig
    unsigned long long* build_stat;   // [2] device: raggedness sums of k_build_lists
    int4* posq;              // [n] sorted: quantised x,y,z (units of L/2^32) + type
    int4* posq_build;        // [n] copy at the last build (displacement check)
    unsigned* cell_of;       // [n] orig: cell id        (build scratch)
    unsigned* rank_in_cell;  // [n] orig                 (build scratch)
    int* order_tmp;          // [n]                      (build scratch)
    unsigned* cell_count;    // [n_cells + 1]
    unsigned* cell_start;    // [n_cells + 1]
    unsigned* scan_tmp;      // block totals
    int64_t cell_cap, scan_cap;

    int capA, capS;          // allocated rows
    int* listA;  int* cntA;  // [capA][n] sorted indices with |r| < rcA + skin
    int* listS;  int* cntS;  // [capS][n] rcA + skin <= |r| < rcR + skin
    int* listT;              // [n][capA+capS] atom-major copy of both lists (reverse-index search): build scratch, in pf's storage if it fits
    int* listT_own;          // ... its own allocation otherwise
    unsigned char* rev;      // [capA][n] slot of i in j's listA
    unsigned char* revS;     // [capS][n] slot of i in j's listS
    int* cA; int* ncA;       // [capA][n] per step: packed (j<<8)|(slot of i in j's skin list) with |r| < rcA
    unsigned long long* mask;   // [n][mrec] per step: in-cutoff masks over the skin slots (see k_filter)
    int64_t mask_cap;           // allocated 64-bit words
    int* cB; int* ncB;       // [capA+capS][n] per step: packed like cA, rcA <= |r| < rcR (listA part, then listS part)
    int* flags;              // [4] device: 0 overflow A, 1 overflow S, 2 max cntA, 3 max (cntA+cntS)
    unsigned* disp_max;      // [2] device: float bits of the max displacement^2 since the build: [0] at the last evaluation, [1] at any evaluation since
    int64_t atom_cap;        // allocated atoms

    float* q;                // [D][n]
    float* fp;               // [D][n]
    float* S;                // [NA*24][n]
    float* U;                // [n]
    float4* pf;              // [capA][n] received from j = cA[m][i]: angular dU_j/dr_ji
    float* mA;               // [capA][n] received from j = cA[m][i]: radial scalar m_ji
    float* mB;               // [capA+capS][n] received from j = cB[m][i]: radial scalar m_ji
    float4* fa;              // [n] sum_j dU_i/dr_ij (angular part from k_force_angular, radial added by k_force_radial)
    double* e_out;           // [n]    orig order
    double* f_out;           // [n][3]
    double* w_out;           // [n][9]

    double* thermo;          // [blocks] partials of sum m v^2, then {lambda, T before the rescale} of the last step
    int thermo_cap;
    double* loss_partial;    // [11 * blocks + 11] block partials and totals of nep_loss_terms
    int loss_cap;
    double* heat_partial;    // [3 * blocks + 3] block partials of the total heat current (nep_heat_current)
    int heat_cap;

    // staging of the host-buffer entry points (device copies of the caller's host arrays)
    double* h_pos; double* h_vel; int* h_type;
    int64_t h_cap;
    bool h_run;              // an md_run_host trajectory is in progress (continuation allowed)
    cudaStream_t copy_stream;   // md_run_host: second stream for the position download (created on first use)
    cudaEvent_t ev_pos;         // ... recorded when the positions of the last step are final

    // batched evaluation for training (nep_batch.cuh): structures concatenated, lattice-image neighbour entries
    struct {
        int n_str, N, cap;                 // structures, atoms of the batch, storage slots per atom
        int* off; int* sid; int* M;        // [n_str+1] atom offsets, [N] structure of an atom, [n_str][3] image reach
        double* H; double* Hinv;           // [n_str][9]
        int* type;                         // [N]
        int* cnt; int* cntA; int* nbr;     // [N] entries, [N] of which inside rc_angular (stored first), [N][cap]
        float4* d;                         // [N][cap] pair vector + distance
        unsigned short* code; unsigned short* rev;   // [N][cap] image-shift code, slot of the reverse entry
        unsigned char* tnb;                // [N][cap] type of the entry's neighbour
        int* bad;                          // [1] device flag
        float* par[6]; size_t par_cap[6];  // parameters of all members of a call
        float* q; float* S; float* fp; float4* pf; size_t scratch_rows;   // per (member, atom) scratch of a chunk
        double* loss_part; size_t loss_cap;
    } b;

    // bookkeeping of owned device memory (nep_device_bytes)
    struct { void* p; size_t bytes; } owned[160];
    int n_owned;
};

// ---------------------------------------------------------------------------------------------------
#define NEP_CUDA(call)                                                                              \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess) {                                                                    \
            snprintf(nep->err, sizeof(nep->err), "%s:%d: %s: %s", __FILE__, __LINE__, #call,        \
                     cudaGetErrorString(e_));                                                       \
            return NEP_ERR_CUDA;                                                                    \
        }                                                                                           \
    } while (0)

#define NEP_LAUNCH_CHECK()                                                                          \
    do {                                                                                            \
        nep->launches++;                                                                            \
        cudaError_t e_ = cudaGetLastError();                                                        \
        if (e_ != cudaSuccess) {                                                                    \
            snprintf(nep->err, sizeof(nep->err), "%s:%d: launch: %s", __FILE__, __LINE__,           \
                     cudaGetErrorString(e_));                                                       \
            return NEP_ERR_CUDA;                                                                    \
        }                                                                                           \
    } while (0)

// Drains the recorded event pairs into prof_ms / prof_n (synchronises the stream).
static inline void nep_prof_drain(nep_t* nep)
{
    if (!nep->prof_ev || nep->prof_used == 0) return;
    cudaEventSynchronize(nep->prof_ev[2 * (nep->prof_used - 1) + 1]);
    for (int p = 0; p < nep->prof_used; ++p) {
        float ms = 0.0f;
        if (cudaEventElapsedTime(&ms, nep->prof_ev[2 * p], nep->prof_ev[2 * p + 1]) == cudaSuccess) {
            nep->prof_ms[nep->prof_kid[p]] += (double)ms;
            nep->prof_n[nep->prof_kid[p]] += 1;
        }
    }
    cudaGetLastError();
    nep->prof_used = 0;
}

static inline void nep_prof_begin(nep_t* nep, int kid)
{
    if (!nep->prof_on) return;
    if (nep->prof_used == NEP_PROF_PAIRS) nep_prof_drain(nep);
    nep->prof_kid[nep->prof_used] = kid;
    cudaEventRecord(nep->prof_ev[2 * nep->prof_used], nep->stream);
}

static inline void nep_prof_end(nep_t* nep)
{
    if (!nep->prof_on) return;
    cudaEventRecord(nep->prof_ev[2 * nep->prof_used + 1], nep->stream);
    nep->prof_used++;
}

// NEP_LAUNCH(kernel id, kernel<<<...>>>(...)): launch + error check (+ event pair when profiling)
#define NEP_LAUNCH(kid, ...)                                                                        \
    do {                                                                                            \
        nep_prof_begin(nep, (kid));                                                                 \
        __VA_ARGS__;                                                                                \
        nep_prof_end(nep);                                                                          \
        NEP_LAUNCH_CHECK();                                                                         \
    } while (0)

static inline int nep_fail(nep_t* nep, int status, const char* msg)
{
    if (nep) snprintf(nep->err, sizeof(nep->err), "%s", msg);
    return status;
}

static inline int div_up(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }
static inline int round_up4(int a) { return (a + 3) & ~3; }
__device__ __forceinline__ int round_up4_dev(int a) { return (a + 3) & ~3; }

// ---------------------------------------------------------------------------------------------------
// Pair geometry from quantised coordinates.  Positions are stored as 32-bit fractions along the lattice
// vectors a, b, c, so the wrapped integer difference IS the minimum image (exact, branch-free; reading A8t:
// valid for cutoffs up to half the smallest perpendicular width); it is converted to Angstrom in fp32,
// d = fa a + fb b + fc c -- one multiplication per component in an orthorhombic cell.  d = r_j - r_i.  dx(i,j) = -dx(j,i) bit for bit, so r2 is the same
// for both orderings of a pair and both atoms take the same in-cutoff decision.
__device__ __forceinline__ void pair_vec(const int4& pi, const int4& pj, const NepDims& D,
                                         float& dx, float& dy, float& dz, float& r2)
{
    const float fa = (float)(int)((unsigned)pj.x - (unsigned)pi.x);
    const float fb = (float)(int)((unsigned)pj.y - (unsigned)pi.y);
    const float fc = (float)(int)((unsigned)pj.z - (unsigned)pi.z);
    if (!D.tri) { dx = fa * D.h[0]; dy = fb * D.h[4]; dz = fc * D.h[8]; }
    else {
        dx = fmaf(fc, D.h[6], fmaf(fb, D.h[3], fa * D.h[0]));
        dy = fmaf(fc, D.h[7], fmaf(fb, D.h[4], fa * D.h[1]));
        dz = fmaf(fc, D.h[8], fmaf(fb, D.h[5], fa * D.h[2]));
    }
    r2 = dx * dx + dy * dy + dz * dz;
}

// Cutoff function Eq. (5) and the Chebyshev argument of Eq. (4).
// f_k(r) = 1/2 [T_k(x)+1] f_c(r), x = 2 (r/rc - 1)^2 - 1.  The recurrence state is advanced by the
// caller: T_{k+1} = 2 x T_k - T_{k-1};  T_k' = k U_{k-1}, U_{k+1} = 2 x U_k - U_{k-1}.
struct BasisHead {
    float x, two_x;       // Chebyshev argument
    float hfc;            // f_c / 2
    float hdfc;           // f_c' / 2
    float hfc_dx;         // (f_c / 2) * dx/dr
};

// f_c needs cos(pi t), f_c' needs sin(pi t), t = r/rc in [0,1).  With u = t - 1/2 in [-1/2, 1/2):
// cos(pi t) = -sin(pi u), sin(pi t) = cos(pi u); both by minimax polynomials in u^2 (degree 9 / 10, error
// < 1e-8 before rounding -- as good as fp32 allows), constants 1/4 and -pi/4 folded into the coefficients.
template <bool WITH_DERIV>
__device__ __forceinline__ BasisHead basis_head(float r, float rc_inv)
{
    BasisHead b;
    const float t = r * rc_inv;
    const float y = t - 1.0f;
    b.x = fmaf(2.0f * y, y, -1.0f);
    b.two_x = 2.0f * b.x;
    const float u = t - 0.5f, v = u * u;
    float ps = fmaf(1.941441508e-02f, v, -1.495728214e-01f);       // sin(pi u) / (4 u)
    ps = fmaf(ps, v, 6.375193808e-01f);
    ps = fmaf(ps, v, -1.291927521e+00f);
    ps = fmaf(ps, v, 7.853981600e-01f);
    b.hfc = fmaf(-u, ps, 0.25f);                                   // (1 + cos(pi t)) / 4
    if (WITH_DERIV) {
        float pc = fmaf(1.916082836e-02f, v, -1.845193348e-01f);   // -(pi/4) cos(pi u)
        pc = fmaf(pc, v, 1.048673055e+00f);
        pc = fmaf(pc, v, -3.187702720e+00f);
        pc = fmaf(pc, v, 3.875784535e+00f);
        pc = fmaf(pc, v, -7.853981632e-01f);
        b.hdfc = pc * rc_inv;                                      // -(pi / 4 rc) sin(pi t)
        b.hfc_dx = b.hfc * (4.0f * y * rc_inv);
    } else {
        b.hdfc = 0.0f;
        b.hfc_dx = 0.0f;
    }
    return b;
}
