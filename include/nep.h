/*
 * nep.h -- C ABI of the B200-native NEP3 hot path (arxiv 2205.10046: Fan et al., GPUMD / NEP3).
 *
 * One handle = one model on one GPU and one CUDA stream.  All work of every call is enqueued on the
 * stream given to nep_create(); a call synchronises that stream only where stated.  Pointers named
 * *_dev are caller-owned DEVICE memory (e.g. torch tensors' data_ptr()) valid for the duration of the
 * call; pointers named *_host (and all parameter arrays of nep_create) are HOST memory.  The handle
 * owns only its internal scratch (neighbour lists, descriptor sums, partial forces, quantised
 * positions), sized at nep_neighbors() and reused.
 *
 * Units: eV, Angstrom, amu, fs.  Atom order of every output is the caller's atom order (the internal
 * spatial sort is invisible).  Every function returns NEP_OK (0) or a negative nep_status;
 * nep_last_error() gives a text for the last failure on that handle.  There is no CPU fallback: every
 * step runs in the library's CUDA kernels, and every entry point except nep_num_descriptors() and
 * nep_status_string() fails with NEP_ERR_CUDA when no CUDA device is usable.
 *
 * Citations are to /root/reference/PAPER.md (line numbers) and to DESIGN.md "Readings" for the places
 * where the paper is silent or garbled.
 */
#ifndef NEP_B200_H_
#define NEP_B200_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nep_ctx nep_t;

/* Hyper-parameters of a NEP3 model in the paper's notation (the keywords of nep.in).   */
typedef struct {
    int32_t n_types;                        /* N_typ >= 1; at most 16                   */
    double rc_radial, rc_angular;           /* r_c^R, r_c^A in Angstrom; 0 < rc_angular <= rc_radial  */
    int32_t n_max_radial, n_max_angular;    /* n = 0..n_max; 0..15 / 0..15       */
    int32_t basis_radial, basis_angular;    /* N_bas: k = 0..N_bas; 0..31            */
    int32_t l_max_3b;                       /* must be 4 (Eqs. 13-16)               */
    int32_t l_max_4b;                       /* 0 (no 4-body block) or 2                */
    int32_t l_max_5b;                       /* 0 (no 5-body block) or 1                */
    int32_t n_neurons;                      /* N_neu >= 1 (Eq. 1); at most 200        */
} nep_hyper_t;

typedef enum {
    NEP_OK = 0,
    NEP_ERR_INVALID_ARG = -1,        /* null pointer, value out of the ranges above, n <= 0, cap too small */
    NEP_ERR_BOX_TOO_SMALL = -2,      /* a perpendicular width < 2 (rc_radial + skin): minimum image breaks */
    NEP_ERR_UNSUPPORTED_BOX = -3,    /* degenerate or left-handed cell (det of the row vectors <= 0)      */
    NEP_ERR_NEIGHBOR_OVERFLOW = -4,  /* a list outgrew its storage and regrowing failed (never truncated) */
    NEP_ERR_STATE = -5,              /* compute / md_step before nep_neighbors, or hook before compute    */
    NEP_ERR_CUDA = -6,               /* a CUDA runtime call failed (text in nep_last_error)               */
    NEP_ERR_NOMEM = -7,              /* device or host allocation failed                                  */
    NEP_ERR_SKIN_EXCEEDED = -8       /* md_step*: an atom moved more than skin/2 between two list builds   */
} nep_status;

/* ---- model ---------------------------------------------------------------------------------------
 * nep_create: builds a handle; copies all parameter arrays (HOST, fp32) to the device.  Synchronises.
 *   c_radial  [T][T][NR][KR]  c^{ij}_{nk} of Eq. (3), index (t_i, t_j, n, k); t_i = type of
 *                             the central atom i, t_j = type of the neighbour; NOT assumed symmetric.
 *   c_angular [T][T][NA][KA]  same for the angular radial functions.
 *   w0 [H][D] row-major ([neuron][descriptor], Listing 1), b0 [H], w1 [H], b1 [1]:
 *             U = sum_m w1[m] tanh(sum_v w0[m][v] q_v - b0[m]) - b1   (Eq. 1).
 *   mass_amu  [T] masses per type (used by md_step only).
 *   NR = n_max_radial+1, KR = basis_radial+1, NA = n_max_angular+1, KA = basis_angular+1,
 *   D = nep_num_descriptors(h), H = n_neurons.
 *   Descriptor order (reading A2): v = n for the radial components (Eq. 2); then the blocks
 *   l = 1,2,3,4 (Eqs. 13-16), 4-body q_n222 (Eq. 18), 5-body q_n1111 (Eq. 19): v = NR + block*NA + n.
 *   device: CUDA device ordinal; cuda_stream: a cudaStream_t (NULL = the legacy default stream).
 * nep_destroy: synchronises the stream and frees everything the handle owns.                          */
int nep_create(nep_t** out, const nep_hyper_t* h,
               const float* c_radial, const float* c_angular,
               const float* w0, const float* b0, const float* w1, const float* b1,
               const double* mass_amu, int device, void* cuda_stream);
int nep_destroy(nep_t* nep);

/* N_des of Eq. (20); pure host arithmetic; negative status on invalid h.           */
int nep_num_descriptors(const nep_hyper_t* h);

/* ---- (a1) neighbour construction -----------------------------------------------------------------
 * Cell-binned construction of the radial and angular neighbour lists NN^R/NL^R, NN^A/NL^A
 * (construction itself is not described by the paper).
 *   pos_dev  [n][3] fp64 positions (need not be wrapped into the box);  type_dev [n] int32 in [0,T);
 *   box      HOST, 9 doubles: the cell's lattice vectors a, b, c as rows (Angstrom), right-handed
 *            (det > 0); orthorhombic or general (triclinic).  Every perpendicular width of the cell must
 *            be >= 2 (rc_radial + skin) (NEP_ERR_BOX_TOO_SMALL), so that the minimum image is unique;
 *   skin     >= 0: lists hold every pair with |r_ij| < r_c + skin (Verlet skin).
 * Membership.  Orthorhombic cell (all off-diagonal elements zero), reading A8: with
 * d = (r_j - r_i) - L*rint((r_j - r_i)/L) per axis in IEEE fp64, j is a neighbour of i iff
 * (dx*dx + dy*dy) + dz*dz < (r_c+skin)*(r_c+skin).  General cell, reading A8t: t = r_j - r_i,
 * n_k = rint((t_x Hinv[x][k] + t_y Hinv[y][k]) + t_z Hinv[z][k]), d = ((t - n_a a) - n_b b) - n_c c, same
 * test.  Both are evaluated exactly so (fp64, no contraction) for every candidate near a cutoff, so
 * the sets equal a brute-force fp64 search bit for bit.  The list order within an atom is unspecified
 * but deterministic.  Copies the types; synchronises (reads back list sizes; regrows and rebuilds on
 * overflow; NEP_ERR_INVALID_ARG if a type is outside [0, T)).  n <= 16,777,216 = 2^24 (list entries pack the
 * neighbour's index into 24 bits; tests/test_gpu_fullsize.py runs exactly 2^24 atoms).                 */
int nep_neighbors(nep_t* nep, int64_t n, const double* pos_dev, const int32_t* type_dev,
                  const double box[9], double skin);

/* Largest list length of the last build: which = 0 radial (r_c^R + skin), 1 angular (r_c^A + skin).   */
int nep_max_neighbors(nep_t* nep, int which, int32_t* max_count_host);

/* Copies the lists of the last build out in the caller's atom order and numbering:
 * count_dev [n], list_dev [n][cap] row-major (entries m >= count are left untouched).
 * NEP_ERR_INVALID_ARG if cap < nep_max_neighbors().  Does not synchronise.                            */
int nep_get_neighbors(nep_t* nep, int which, int32_t* count_dev, int32_t* list_dev, int32_t cap);

/* ---- (a2)-(a8) energy, force, virial -------------------------------------------------------------
 * One evaluation with the lists of the last nep_neighbors() (valid while no atom has moved more than
 * skin/2 since then): Chebyshev radial descriptors Eqs. (2)-(5); angular sums S_nk Eq. (12) and the
 * 3-/4-/5-body components Eqs. (13)-(19); network Eq. (1); partial forces Eq. (21); F_i Eqs. (22)-(23);
 * per-atom virial W_i Eq. (24).
 *   pos_dev    [n][3] fp64;
 *   energy_dev [n] fp64 site energies U_i (eV);  force_dev [n][3] fp64 (eV/Angstrom);
 *   virial_dev [n][9] fp64 (eV), W[3a+b] = sum_j r_ij^a (dU_j/dr_ji)^b, r_ij = r_j - r_i (not symmetrised;
 *              sum_i W_i = -dE/d(strain), reading A7).   Any output pointer may be NULL.
 * Arithmetic: fp32 inside the kernels, fp64 I/O.  Does not synchronise.                */
int nep_compute(nep_t* nep, const double* pos_dev, double* energy_dev, double* force_dev, double* virial_dev);

/* ---- (a9) velocity-Verlet NVE ---------------------------------------------------------------------
 * n_steps steps of  v += (dt/2) F/m;  r += dt v;  [lists rebuilt when the number of steps since the
 * last build reaches rebuild_every];  F = F(r);  v += (dt/2) F/m   (NVE; the paper prints no
 * integrator formula, reading A11).  a[A/fs^2] = F/m * 9.648533212e-3.
 *   pos_dev [n][3], vel_dev [n][3] (Angstrom/fs) are updated in place; positions are never wrapped.
 *   The first call after nep_neighbors()/nep_compute() with other positions evaluates F(r) first; later
 *   calls reuse the forces of the previous call (so positions must not be edited in between without
 *   calling nep_neighbors() again).  rebuild_every >= 1; skin as in nep_neighbors().
 * Skin check (all md_step* calls): the lists are valid while no atom has moved more than skin/2 since the
 * build.  The largest displacement of every evaluation is reduced on the device; it is read at every
 * scheduled rebuild and when the call ends, and NEP_ERR_SKIN_EXCEEDED is returned if it was ever above
 * skin/2 (pairs may then have been missed since that build: use a smaller rebuild_every or a larger skin;
 * the state in pos_dev / vel_dev is the one reached, not rolled back).  At a scheduled rebuild the check
 * comes BEFORE the rebuild, so a skin error is never hidden by an error of that rebuild.
 * The criterion is sufficient, not necessary: it bounds every atom's ABSOLUTE displacement, so a rigid
 * translation or a net centre-of-mass drift larger than skin/2 per interval is reported although no pair
 * distance changed (remove the centre-of-mass velocity, or rebuild more often).  nep_compute() with moved
 * positions measures the same displacement but checks nothing: such callers poll nep_max_displacement().
 * Synchronises once per list rebuild (overflow check) and once before it returns (skin check).        */
int md_step(nep_t* nep, double* pos_dev, double* vel_dev, double dt_fs,
            int32_t n_steps, int32_t rebuild_every, double skin);

/* ---- NVT: velocity-Verlet + Berendsen thermostat (named PAPER.md:318, `nvt_ber` PAPER.md:602, ref. 75;
 * equation per DESIGN.md reading A15).  As md_step, and after the second half kick of every step all
 * velocities are scaled by lambda = sqrt(1 + (dt_fs / tau_fs) (T_target / T - 1)), T = sum m v^2 / (3 n k_B),
 * T_target of step s = 1..n_steps = t_start_K + (t_stop_K - t_start_K) s / n_steps.  The kinetic-energy sum
 * is reduced on the device in a fixed order; no host round trip.  NEP_ERR_INVALID_ARG if tau_fs < dt_fs (the
 * rescale would overshoot the target; lambda^2 is clamped at 0 besides), tau_fs <= 0 or a temperature < 0.  nep_last_temperature: T before the rescale and lambda of the last thermostatted step
 * (host scalars; synchronises; NEP_ERR_STATE if there was none).                                        */
int md_step_nvt_berendsen(nep_t* nep, double* pos_dev, double* vel_dev, double dt_fs, int32_t n_steps,
                          int32_t rebuild_every, double skin, double t_start_K, double t_stop_K, double tau_fs);
int nep_last_temperature(nep_t* nep, double* t_before_host, double* lambda_host);

/* ---- NVT: velocity-Verlet + Langevin thermostat (named PAPER.md:318, `nvt_lan` PAPER.md:574-590, refs.
 * 80-81; equations per DESIGN.md reading A16).  Every MD step s = first_step .. first_step + n_steps - 1 is:
 * thermostat half step, the velocity-Verlet step of md_step, thermostat half step; a half step replaces every
 * velocity component by c1 v + sqrt(1 - c1^2) sqrt(k_B T_target / m) R with c1 = exp(-dt_fs / (2 tau_fs)) and R
 * the counter-based standard normal deviate of reading A16 (seed; counter from the step number, the atom's
 * index in the caller's order and the component), so the random forces are reproducible and independent of how
 * the steps are split over calls (pass first_step = steps done so far).  T_target ramps as in
 * md_step_nvt_berendsen, i.e. over the steps of ONE call: a ramp split over several calls must be split by the
 * caller (t_start_K / t_stop_K of each piece); with t_start_K == t_stop_K the whole trajectory is independent of
 * the split.  NEP_ERR_INVALID_ARG if tau_fs <= 0, a temperature < 0 or first_step < 0.        */
int md_step_nvt_langevin(nep_t* nep, double* pos_dev, double* vel_dev, double dt_fs, int32_t n_steps,
                         int32_t rebuild_every, double skin, double t_start_K, double t_stop_K, double tau_fs,
                         uint64_t seed, int64_t first_step);

/* Results of the most recent internal evaluation (the one md_step ended with, or nep_compute):
 * same layouts as nep_compute; any pointer may be NULL.  Does not synchronise.                        */
int nep_get_last(nep_t* nep, double* energy_dev, double* force_dev, double* virial_dev);

/* Largest displacement (Angstrom) of any atom since the last list build, measured at the most recent
 * evaluation; the lists are valid while it is below skin/2.  Synchronises.                            */
int nep_max_displacement(nep_t* nep, double* disp_host);

/* Measurement support: raggedness of the skin lists of the last build -- the sum over warps (32 consecutive atoms
 * of the internal order) of 32 x the longest list, divided by the sum of all list lengths: the factor by which a
 * pair loop is slowed by idle lanes when a warp's atoms have unequal lists (1.0 in a perfect crystal; it grows as a
 * structure disorders).  NEP_ERR_STATE before nep_neighbors.                            */
int nep_list_raggedness(nep_t* nep, double* raggedness_host);

/* ---- host-buffer entry points (end-to-end path: H2D copies, kernels, D2H copies) -------------------
 * All *_host arrays are HOST memory (pageable or pinned; pinned makes the copies asynchronous DMA).
 * The device staging copies are owned by the handle and reused between calls.  Both synchronise.
 * nep_compute_host: upload pos/type, nep_neighbors + one evaluation, download the non-NULL results.
 * md_run_host: upload pos/vel, run n_steps of md_step, download pos/vel and the non-NULL results of the
 *   final evaluation.  type_host != NULL STARTS a run: types are uploaded and the lists built from the
 *   uploaded positions (box, skin as in nep_neighbors).  type_host == NULL CONTINUES the run the previous
 *   md_run_host call on this handle left (same n): types, lists, rebuild cadence and the forces of the
 *   last evaluation carry over, `box` is ignored; the uploaded positions must be the ones that call
 *   returned (velocities may have been changed, e.g. by a host-side thermostat).  NEP_ERR_STATE if there
 *   is nothing to continue.                                                                            */
int nep_compute_host(nep_t* nep, int64_t n, const double* pos_host, const int32_t* type_host,
                     const double box[9], double skin,
                     double* energy_host, double* force_host, double* virial_host);
int md_run_host(nep_t* nep, int64_t n, double* pos_host, double* vel_host, const int32_t* type_host,
                const double box[9], double dt_fs, int32_t n_steps, int32_t rebuild_every, double skin,
                double* energy_host, double* force_host, double* virial_host);

/* ---- descriptor / latent-vector export and test hooks (last evaluation, caller's atom order) -------
 * nep_get_descriptors: q_dev [n][D] descriptor vector q_i^v of Eq. (1) in the order of DESIGN.md reading
 *   A2 (what PYNEP's 'descriptor' property returns), fp_dev [n][D] dU_i/dq_v
 *   (PAPER.md:901).  nep_get_angular_sums: S_dev [n][NA][24] sums of Eq. (12) (test hook).
 * nep_get_latent: latent_dev [n][H], the latent-space vector of PAPER.md:484 -- component mu is the state
 *   of hidden neuron mu times its weight to the output layer, w1_mu tanh(sum_v w0_mu,v q_v - b0_mu), so
 *   that sum_mu latent[i][mu] - b1 = U_i.
 * All fp32 device buffers owned by the caller; any pointer of the first two calls may be NULL.
 * NEP_ERR_STATE before the first evaluation.  Do not synchronise.                                     */
int nep_get_descriptors(nep_t* nep, float* q_dev, float* fp_dev);
int nep_get_angular_sums(nep_t* nep, float* S_dev);
int nep_get_latent(nep_t* nep, float* latent_dev);

/* ---- parameter sets: SNES training evaluates a POPULATION of parameter vectors z on the same structures
 * (Eqs. (31)-(33)); the neighbour lists and the per-step in-cutoff lists depend on the
 * geometry only (single-structure slice).
 * nep_set_parameters: replaces the model parameters (same hyper-parameters, same layouts as nep_create);
 *   lists stay valid; the next nep_compute / md_step uses the new model.  Synchronises the stream.
 * nep_compute_population: n_pop parameter sets, stacked member-major in HOST arrays (c_radial
 *   [n_pop][T][T][NR][KR], c_angular [n_pop][T][T][NA][KA], w0 [n_pop][H][D], b0, w1 [n_pop][H], b1 [n_pop]),
 *   evaluated at the same positions: energy_dev [n_pop][n], force_dev [n_pop][n][3], virial_dev
 *   [n_pop][n][9] (any may be NULL).  Positions are quantised and the skin lists filtered once; every
 *   member runs the descriptor, network and force kernels.  Leaves the LAST member's parameters in the
 *   handle.  NEP_ERR_STATE before nep_neighbors.  Synchronises once per member (parameter upload).         */
int nep_set_parameters(nep_t* nep, const float* c_radial, const float* c_angular,
                       const float* w0, const float* b0, const float* w1, const float* b1);
int nep_compute_population(nep_t* nep, const double* pos_dev, int32_t n_pop,
                           const float* c_radial, const float* c_angular,
                           const float* w0, const float* b0, const float* w1, const float* b1,
                           double* energy_dev, double* force_dev, double* virial_dev);

/* Data terms of the loss function, Eq. (33) (reading A17), of the LAST evaluation
 * for one structure of n atoms: terms_host[0] = |sum_i U_i / n - u_target_per_atom|, [1] = sqrt(sum_i |F_i -
 * F_i^tar|^2 / (3 n)), [2] = sqrt(sum over {xx,yy,zz,xy,yz,zx} of (sum_i W_i / n - w_target_per_atom)^2 / 6).
 * f_target_dev [n][3] device, w_target_per_atom[6] and terms_host[3] host.  Reduced on the device in a fixed
 * order; synchronises.  The weights lambda and the regularisation terms of Eq. (33) are the caller's.      */
int nep_loss_terms(nep_t* nep, double u_target_per_atom, const double* f_target_dev,
                   const double w_target_per_atom[6], double terms_host[3]);

/* ---- batched evaluation for training: many small structures x a population of parameter sets ------------------
 * (SURVEY.md section 8(f) row 4.)  SNES evaluates every member of a population on every structure of a (mini-)batch
 * and reduces the loss of Eq. (33).  Independent of nep_neighbors()/md_step(): the batch has its
 * own storage in the handle.
 * nep_batch_neighbors: n_str structures concatenated; structure s owns atoms atom_offset_host[s] .. [s+1]-1 (HOST,
 *   [n_str+1], starting at 0, at least one atom each); pos_dev [N][3] fp64 and type_dev [N] int32 (DEVICE), N =
 *   atom_offset_host[n_str]; boxes_host [n_str][9] (HOST): lattice vectors a, b, c of each cell as rows, det > 0.
 *   The cells may be of ANY size > rc_radial / 6.5 per perpendicular width (NEP_ERR_BOX_TOO_SMALL below that):
 *   the neighbours of atom i are all lattice images (j, N) != (i, 0) of the atoms of its own structure with
 *   |r_j + N_a a + N_b b + N_c c - r_i| < rc_radial (angular: < rc_angular), evaluated in fp64 (DESIGN.md reading
 *   A18); positions need not be wrapped.  Synchronises (sizes the storage from the longest list).
 * nep_batch_compute: evaluates n_pop parameter sets (HOST arrays stacked member-major, layouts of nep_create as in
 *   nep_compute_population) on every structure of the batch in one launch sequence over atoms x members; the
 *   parameters are copied to the device once, there is no per-member synchronisation.  energy_dev [n_pop][N]
 *   (required), force_dev [n_pop][N][3], virial_dev [n_pop][N][9] (either may be NULL), fp64, batch atom order.
 *   Does not touch the handle's own model.  Synchronises before returning (the host arrays may then be reused).
 * nep_batch_loss: the three data terms of Eq. (33) for every member, from the outputs of nep_batch_compute and the
 *   targets u_target_dev [n_str] (eV/atom), f_target_dev [N][3] (eV/Angstrom), w_target_dev [n_str][6] (eV/atom;
 *   xx, yy, zz, xy, yz, zx of W[3a+b]):  loss_dev [n_pop][3] = { sqrt(1/n_str sum_s (sum_i U_i/N_s - u_tar_s)^2),
 *   sqrt(1/(3N) sum_i |F_i - F_i^tar|^2), sqrt(1/(6 n_str) sum_s sum_{mu nu} (sum_i W_i/N_s - w_tar_s)^2) },
 *   reduced on the device per (member, structure) and then per member in a fixed order (bitwise reproducible).
 *   The weights lambda and the regularisation terms of Eq. (33) are the caller's.  Does not synchronise.
 * NEP_ERR_STATE before nep_batch_neighbors.                                                                      */
int nep_batch_neighbors(nep_t* nep, int32_t n_str, const int32_t* atom_offset_host, const double* pos_dev,
                        const int32_t* type_dev, const double* boxes_host);
int nep_batch_compute(nep_t* nep, int32_t n_pop, const float* c_radial, const float* c_angular,
                      const float* w0, const float* b0, const float* w1, const float* b1,
                      double* energy_dev, double* force_dev, double* virial_dev);
/* Measurement support: ordered neighbour entries of the batch inside rc_radial and inside rc_angular (lattice images
 * counted), summed over all atoms.  Synchronises.  NEP_ERR_STATE before nep_batch_neighbors.                       */
int nep_batch_pair_counts(nep_t* nep, int64_t* radial_entries_host, int64_t* angular_entries_host);

int nep_batch_loss(nep_t* nep, int32_t n_pop, const double* energy_dev, const double* force_dev,
                   const double* virial_dev, const double* u_target_dev, const double* f_target_dev,
                   const double* w_target_dev, double* loss_dev);

/* ---- heat current, Eqs. (25)-(26) ------------------------------------------------
 * J_i = W_i . v_i with the per-atom virial W_i of the last evaluation (Eq. (24), layout W[3a+b]):
 * j_atom_dev [n][3] gets J_i^a = sum_b W_i^{ab} v_i^b, j_total_dev [3] gets J = sum_i J_i (reduced in a
 * fixed order: bitwise reproducible).  vel_dev [n][3] Angstrom/fs in the caller's atom order, which must be
 * the velocities that belong to the evaluated positions (after md_step: the vel_dev it was given).
 * fp64 device buffers owned by the caller; either output may be NULL, not both.  Units eV Angstrom / fs.
 * NEP_ERR_STATE before the first evaluation.  Does not synchronise.                                    */
int nep_heat_current(nep_t* nep, const double* vel_dev, double* j_atom_dev, double* j_total_dev);

/* nep_heat_current_static: the same J_i and J as nep_heat_current, for callers that must not allocate.
 * Who that is: a sampling loop (Green-Kubo runs read J every few steps) inside a process
 * whose free device memory already belongs to someone else -- a framework's caching allocator, a second
 * simulation sharing the GPU -- so that a cudaMalloc of even a few hundred kB fails; and threads that cannot
 * afford the device-wide stall an allocation or a free may cause for every other stream.  nep_heat_current
 * grows a cudaMalloc'ed scratch buffer for its block partials on first use and when n grows; this call uses
 * a fixed array inside the library image instead and calls no cudaMalloc, cudaFree or any allocating routine.
 *   Limit:  n <= 4,194,304 atoms (the array holds 3 partials per 256 atoms: 393,240 bytes).  Larger systems
 *           return NEP_ERR_INVALID_ARG with a message naming the limit; use nep_heat_current for them.
 *   Cost:   every GPU on which the library is loaded holds those 393,240 bytes until the process exits,
 *           used or not.
 *   Set-up: the FIRST call on each device looks up the array's device address (cudaGetSymbolAddress, with
 *           that device current) and keeps it; make that first call outside any stream capture.
 *   Sharing: all handles and all calls on one device use the same array, and it keeps the last call's
 *           partials.  Nothing in it needs clearing (each call overwrites every element it later reads), but
 *           two calls that overlap on the GPU -- different streams, or different handles on different
 *           streams -- race on it and give wrong totals: keep calls on one device ordered.  With
 *           j_total_dev == NULL the total is left in the array's tail, where the next call overwrites it.
 * Arguments, units, order of the reduction (bitwise the same result as nep_heat_current), error codes and
 * "does not synchronise" are as for nep_heat_current; inputs and outputs stay caller-owned device memory. */
int nep_heat_current_static(nep_t* nep, const double* vel_dev, double* j_atom_dev, double* j_total_dev);

/* ---- measurement support (bench.py) ---------------------------------------------------------------
 * nep_launch_count: kernel launches the handle has enqueued so far (bench.py's gpu_launches).
 * nep_device_bytes: device memory the handle currently owns (model tables, lists, scratch, staging).
 * nep_profile(enable): switches per-kernel timing on/off and clears the totals.  While on, every kernel
 *   launch is bracketed by a CUDA event pair on the handle's stream (no synchronisation added, except a
 *   drain every 32768 launches).  nep_profile_read: synchronises and returns, per kernel id
 *   k < nep_profile_num_kernels(), the summed device time in ms and the number of launches since the
 *   last nep_profile() call; nep_profile_kernel_name(k) names the id ("radial", "force_angular", ...).
 * nep_probe_fp32: runs an FP32 FMA throughput probe (16 independent a = fma(a, m, a) chains per thread, no memory
 *   traffic) on `device`/`cuda_stream` at 2, 4, 6 and 8 blocks per SM and returns the best timed launch in TFLOP/s: the measured
 *   denominator of the ALU roofline.  Synchronises.                                                    */
/* nep_pair_counts: ordered pairs inside r_c^R and inside r_c^A at the last evaluation (the sums of
 *   NN_i^R and NN_i^A without skin): the units of the per-kernel flop counts.  Synchronises. */
int nep_pair_counts(nep_t* nep, int64_t* radial_pairs_host, int64_t* angular_pairs_host);
int64_t nep_launch_count(const nep_t* nep);
int64_t nep_device_bytes(const nep_t* nep);
int nep_profile(nep_t* nep, int enable);
int nep_profile_num_kernels(void);
const char* nep_profile_kernel_name(int k);
int nep_profile_read(nep_t* nep, double* ms_total_host, int64_t* launches_host);
int nep_probe_fp32(int device, void* cuda_stream, double* tflops_host);
/* Unit-test probe: packs (j_host[a], slot_host[a]) into a list entry on the device exactly as the list kernels do
 * ((j << 8) | slot, all 32 bits used) and unpacks it again; HOST arrays of `count` int32 each.  0 <= j < 2^24,
 * 0 <= slot < 256, else NEP_ERR_INVALID_ARG.  Allocates and frees its own device buffer; synchronises.  Lets a cheap
 * test cover j >= 2^23 (sign bit of the packed word) without a 2^24-atom system.                                  */
int nep_probe_entry_roundtrip(int device, int32_t count, const int32_t* j_host, const int32_t* slot_host,
                              int32_t* packed_host, int32_t* j_out_host, int32_t* slot_out_host);

const char* nep_last_error(const nep_t* nep);
const char* nep_status_string(int status);

#ifdef __cplusplus
}
#endif
#endif /* NEP_B200_H_ */
