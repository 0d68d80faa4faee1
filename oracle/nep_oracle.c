/*
 * nep_oracle.c -- plain, slow, fp64 CPU ORACLE of the NEP3 hot path (arxiv 2205.10046, PAPER.md).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
 * header, table or constant generator with the CUDA library in paper_2205_10046_b200/csrc/.
 *
 * It is the method's plain definition written out in the paper's order and notation:
 *   O1  brute-force O(N^2) neighbours, minimum image, exact fp64 predicate (reading A8)
 *   O2  radial descriptor        Eqs. (2)-(5)
 *   O3  angular sums S_nk        Eq. (12)            PAPER.md:124-131 (exponent read as l_k, reading G1)
 *       3-body / 4-body / 5-body Eqs. (13)-(16), (18) last line, (19)
 *   O4  network                  Eq. (1), Listing 1
 *   O5  partial forces           Eq. (21)            PAPER.md:203-208 (derivatives derived, see below)
 *   O6  force / virial sums      Eqs. (22)-(24)
 *   O7  velocity-Verlet NVE      (textbook; the paper lists NVE, without a formula)
 * No blocking, fusion, caching or re-association beyond those definitions.  OpenMP (if enabled) only
 * distributes the independent per-atom loops; every per-atom sum is evaluated serially in list order.
 *
 * Pins (tests/test_oracle_pins.py, tests/test_oracle_physics.py): Eq.(6) Legendre double sum,
 * Eqs.(7)-(8) |A_nlm|^2 with library spherical harmonics, Wigner-3j contractions Eqs.(9)-(11),
 * q_n1111 = (7/15) q_n1^2, cos(k arccos x), N_des worked values 55/77/82, central finite differences
 * for F and for dU/dq, sum F = 0, translation / rotation / permutation invariance, sum W = -dE/d(eps),
 * hand-computed dimer; brute-force neighbours (onep_neighbors and the per-selected-atom onep_neighbors_of) vs
 * scipy's cKDTree and a 125-lattice-image search, orthorhombic and sheared.  Parity of E/F/W against any trained-model number of the paper: UNPINNED
 * (the paper's models and datasets are not available) -- see DESIGN.md.
 *
 * Cells of any size (onep_compute_images, reading A18; the small cells of a training batch, Eq. (33),
 * PAPER.md:267-283): neighbours are all lattice images within the cutoffs.  Pins (tests/test_oracle_derived.py): equals
 * the pinned minimum-image path on a supercell of the same crystal, atom by atom (orthorhombic, sheared, and 4-atom
 * cells where atoms see their own images); entry counts vs a numpy lattice-image search; F = -dE/dr and
 * sum W = -dE/d(eps) by central differences in a cell with self-images.
 *
 * Compile: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC nep_oracle.c -o libnep_oracle.so -lm
 * (-ffp-contract=off so that the neighbour predicate is the literal IEEE expression of reading A8).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NUM_B 24

typedef struct {
    int32_t n_types;
    double rc_radial, rc_angular;
    int32_t n_max_radial, n_max_angular;   /* n = 0..n_max */
    int32_t basis_radial, basis_angular;   /* k = 0..N_bas      */
    int32_t l_max_3b, l_max_4b, l_max_5b;  /* 4, {0,2}, {0,1}   */
    int32_t n_neurons;
} onep_hyper;

static const int L_OF_K[NUM_B] = {1,1,1, 2,2,2,2,2, 3,3,3,3,3,3,3, 4,4,4,4,4,4,4,4,4};

int onep_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- counting formula, Eq. (20) PAPER.md:192-197 ------------------------------------------------ */
static int n_blocks(const onep_hyper* h)
{
    return h->l_max_3b + (h->l_max_4b >= 2 ? 1 : 0) + (h->l_max_5b >= 1 ? 1 : 0);
}
int onep_num_descriptors(const onep_hyper* h)
{
    return (h->n_max_radial + 1) + (h->n_max_angular + 1) * n_blocks(h);
}

/* ---- cutoff function Eq. (5) PAPER.md:75 and its derivative ------------------------------------- */
double onep_fc(double r, double rc)
{
    return (r <= rc) ? 0.5 * (1.0 + cos(M_PI * r / rc)) : 0.0;
}
double onep_dfc(double r, double rc)
{
    return (r <= rc) ? -0.5 * (M_PI / rc) * sin(M_PI * r / rc) : 0.0;
}

/* ---- basis functions Eq. (4) PAPER.md:70 --------------------------------------------------------
 * f_k(r) = 1/2 [T_k(x) + 1] f_c(r),  x = 2 (r/rc - 1)^2 - 1,  k = 0..nbas.
 * T_k by T_0 = 1, T_1 = x, T_{k+1} = 2 x T_k - T_{k-1};  T_k' = k U_{k-1}, U_0 = 1, U_1 = 2x,
 * U_{k+1} = 2 x U_k - U_{k-1}.  f_k' = 1/2 [T_k'(x) x'(r) f_c + (T_k + 1) f_c'],  x' = 4 (r/rc - 1)/rc. */
void onep_fk(double r, double rc, int nbas, double* f, double* df)
{
    double x = 2.0 * (r / rc - 1.0) * (r / rc - 1.0) - 1.0;
    double dx = 4.0 * (r / rc - 1.0) / rc;
    double fc = onep_fc(r, rc), dfc = onep_dfc(r, rc);
    double Tkm1 = 1.0, Tk = x;      /* T_0, T_1 */
    double Ukm1 = 0.0, Uk = 1.0;    /* U_{-1} := 0, U_0 */
    for (int k = 0; k <= nbas; ++k) {
        double T, dT;
        if (k == 0) { T = 1.0; dT = 0.0; }
        else if (k == 1) { T = x; dT = 1.0; }
        else {
            double Tn = 2.0 * x * Tk - Tkm1;   /* T_k from T_{k-1}=Tk, T_{k-2}=Tkm1 */
            double Un = 2.0 * x * Uk - Ukm1;   /* U_{k-1} from U_{k-2}=Uk, U_{k-3}=Ukm1 */
            Tkm1 = Tk; Tk = Tn; Ukm1 = Uk; Uk = Un;
            T = Tk; dT = (double)k * Uk;
        }
        f[k] = 0.5 * (T + 1.0) * fc;
        if (df) df[k] = 0.5 * (dT * dx * fc + (T + 1.0) * dfc);
    }
}

/* ---- the 24 polynomials b_k of Eq. (12), PAPER.md:129-131 (b_13 restored, reading G3) -----------
 * written with r^2 = x^2+y^2+z^2 exactly as the paper prints them; homogeneous of degree l_k.      */
void onep_bk(const double d[3], double b[NUM_B])
{
    double x = d[0], y = d[1], z = d[2];
    double r2 = x * x + y * y + z * z;
    b[0] = z;  b[1] = x;  b[2] = y;
    b[3] = 3.0 * z * z - r2;  b[4] = x * z;  b[5] = y * z;  b[6] = x * x - y * y;  b[7] = 2.0 * x * y;
    b[8] = (5.0 * z * z - 3.0 * r2) * z;
    b[9] = (5.0 * z * z - r2) * x;
    b[10] = (5.0 * z * z - r2) * y;
    b[11] = (x * x - y * y) * z;
    b[12] = 2.0 * x * y * z;
    b[13] = (x * x - 3.0 * y * y) * x;
    b[14] = (3.0 * x * x - y * y) * y;
    b[15] = (35.0 * z * z - 30.0 * r2) * z * z + 3.0 * r2 * r2;
    b[16] = (7.0 * z * z - 3.0 * r2) * x * z;
    b[17] = (7.0 * z * z - 3.0 * r2) * y * z;
    b[18] = (7.0 * z * z - r2) * (x * x - y * y);
    b[19] = (7.0 * z * z - r2) * 2.0 * x * y;
    b[20] = (x * x - 3.0 * y * y) * x * z;
    b[21] = (3.0 * x * x - y * y) * y * z;
    b[22] = (x * x - y * y) * (x * x - y * y) - 4.0 * x * x * y * y;
    b[23] = 4.0 * (x * x - y * y) * x * y;
}

/* gradients of the same polynomials with respect to (x,y,z) (derived by hand; pinned by finite
 * differences of onep_bk and, through the forces, by F = -dE/dr).                                  */
void onep_bk_grad(const double d[3], double g[NUM_B][3])
{
    double x = d[0], y = d[1], z = d[2];
    double x2 = x * x, y2 = y * y, z2 = z * z;
#define SETG(k, gx, gy, gz) do { g[k][0] = (gx); g[k][1] = (gy); g[k][2] = (gz); } while (0)
    SETG(0, 0.0, 0.0, 1.0);
    SETG(1, 1.0, 0.0, 0.0);
    SETG(2, 0.0, 1.0, 0.0);
    SETG(3, -2.0 * x, -2.0 * y, 4.0 * z);
    SETG(4, z, 0.0, x);
    SETG(5, 0.0, z, y);
    SETG(6, 2.0 * x, -2.0 * y, 0.0);
    SETG(7, 2.0 * y, 2.0 * x, 0.0);
    SETG(8, -6.0 * x * z, -6.0 * y * z, -3.0 * (x2 + y2 - 2.0 * z2));
    SETG(9, -3.0 * x2 - y2 + 4.0 * z2, -2.0 * x * y, 8.0 * x * z);
    SETG(10, -2.0 * x * y, -x2 - 3.0 * y2 + 4.0 * z2, 8.0 * y * z);
    SETG(11, 2.0 * x * z, -2.0 * y * z, x2 - y2);
    SETG(12, 2.0 * y * z, 2.0 * x * z, 2.0 * x * y);
    SETG(13, 3.0 * (x2 - y2), -6.0 * x * y, 0.0);
    SETG(14, 6.0 * x * y, 3.0 * (x2 - y2), 0.0);
    SETG(15, 12.0 * x * (x2 + y2 - 4.0 * z2), 12.0 * y * (x2 + y2 - 4.0 * z2),
             -16.0 * z * (3.0 * x2 + 3.0 * y2 - 2.0 * z2));
    SETG(16, -z * (9.0 * x2 + 3.0 * y2 - 4.0 * z2), -6.0 * x * y * z, -3.0 * x * (x2 + y2 - 4.0 * z2));
    SETG(17, -6.0 * x * y * z, -z * (3.0 * x2 + 9.0 * y2 - 4.0 * z2), -3.0 * y * (x2 + y2 - 4.0 * z2));
    SETG(18, -4.0 * x * (x2 - 3.0 * z2), 4.0 * y * (y2 - 3.0 * z2), 12.0 * z * (x2 - y2));
    SETG(19, -2.0 * y * (3.0 * x2 + y2 - 6.0 * z2), -2.0 * x * (x2 + 3.0 * y2 - 6.0 * z2), 24.0 * x * y * z);
    SETG(20, 3.0 * z * (x2 - y2), -6.0 * x * y * z, x * (x2 - 3.0 * y2));
    SETG(21, 6.0 * x * y * z, 3.0 * z * (x2 - y2), y * (3.0 * x2 - y2));
    SETG(22, 4.0 * x * (x2 - 3.0 * y2), -4.0 * y * (3.0 * x2 - y2), 0.0);
    SETG(23, 4.0 * y * (3.0 * x2 - y2), 4.0 * x * (x2 - 3.0 * y2), 0.0);
#undef SETG
}

/* ---- pre-computed coefficients, written as the fractions the paper prints ------------------------
 * C^3b: Eqs. (13)-(16) PAPER.md:133-153; C^4b: Eq. (18); C^5b: Eq. (19) */
void onep_constants(double c3[NUM_B], double c4[5], double c5[3])
{
    const double pi = M_PI;
    c3[0] = (1.0 / 4.0) * (3.0 / pi);
    c3[1] = c3[2] = 2.0 * (1.0 / 4.0) * (3.0 / (2.0 * pi));
    c3[3] = (1.0 / 16.0) * (5.0 / pi);
    c3[4] = c3[5] = 2.0 * (1.0 / 4.0) * (15.0 / (2.0 * pi));
    c3[6] = c3[7] = 2.0 * (1.0 / 16.0) * (15.0 / (2.0 * pi));
    c3[8] = (1.0 / 16.0) * (7.0 / pi);
    c3[9] = c3[10] = 2.0 * (1.0 / 64.0) * (21.0 / pi);
    c3[11] = c3[12] = 2.0 * (1.0 / 16.0) * (105.0 / (2.0 * pi));
    c3[13] = c3[14] = 2.0 * (1.0 / 64.0) * (35.0 / pi);
    c3[15] = (9.0 / 256.0) * (1.0 / pi);
    c3[16] = c3[17] = 2.0 * (9.0 / 64.0) * (5.0 / pi);
    c3[18] = c3[19] = 2.0 * (9.0 / 64.0) * (5.0 / (2.0 * pi));
    c3[20] = c3[21] = 2.0 * (9.0 / 64.0) * (35.0 / pi);
    c3[22] = c3[23] = 2.0 * (9.0 / 256.0) * (35.0 / (2.0 * pi));
    {
        double y20 = 0.25 * sqrt(5.0 / pi);            /* (1/4) sqrt(5/pi)      */
        double y21 = 0.5 * sqrt(15.0 / (2.0 * pi));    /* (1/2) sqrt(15/(2 pi)) */
        double y22 = 0.25 * sqrt(15.0 / (2.0 * pi));   /* (1/4) sqrt(15/(2 pi)) */
        c4[0] = -sqrt(2.0 / 35.0) * y20 * y20 * y20;
        c4[1] = -6.0 * sqrt(1.0 / 70.0) * y20 * y21 * y21;
        c4[2] = 6.0 * sqrt(2.0 / 35.0) * y20 * y22 * y22;
        c4[3] = 6.0 * sqrt(3.0 / 35.0) * y21 * y21 * y22;
        c4[4] = -12.0 * sqrt(3.0 / 35.0) * y21 * y21 * y22;
    }
    c5[0] = 21.0 / (80.0 * pi * pi);
    c5[1] = 21.0 / (40.0 * pi * pi);
    c5[2] = 21.0 / (80.0 * pi * pi);
}

/* ---- angular descriptor components of one n from its 24 sums S_k ---------------------------------
 * out[0..3] = q_n1..q_n4 (Eqs. 13-16), out[4] = q_n222 (Eq. 18 last line), out[5] = q_n1111 (Eq. 19).
 * dq[b][k] = d out[b] / d S_k (needed for Eq. (21)).                                                */
void onep_q_from_S(const double S[NUM_B], double out[6], double dq[6][NUM_B])
{
    double c3[NUM_B], c4[5], c5[3];
    onep_constants(c3, c4, c5);
    if (dq) memset(dq, 0, sizeof(double) * 6 * NUM_B);
    for (int b = 0; b < 6; ++b) out[b] = 0.0;
    for (int k = 0; k < NUM_B; ++k) {
        int l = L_OF_K[k];
        out[l - 1] += c3[k] * S[k] * S[k];
        if (dq) dq[l - 1][k] = 2.0 * c3[k] * S[k];
    }
    {
        double s3 = S[3], s4 = S[4], s5 = S[5], s6 = S[6], s7 = S[7];
        out[4] = c4[0] * s3 * s3 * s3 + c4[1] * s3 * (s4 * s4 + s5 * s5) + c4[2] * s3 * (s6 * s6 + s7 * s7)
               + c4[3] * s6 * (s5 * s5 - s4 * s4) + c4[4] * s4 * s5 * s7;
        if (dq) {
            dq[4][3] = 3.0 * c4[0] * s3 * s3 + c4[1] * (s4 * s4 + s5 * s5) + c4[2] * (s6 * s6 + s7 * s7);
            dq[4][4] = 2.0 * c4[1] * s3 * s4 - 2.0 * c4[3] * s6 * s4 + c4[4] * s5 * s7;
            dq[4][5] = 2.0 * c4[1] * s3 * s5 + 2.0 * c4[3] * s6 * s5 + c4[4] * s4 * s7;
            dq[4][6] = 2.0 * c4[2] * s3 * s6 + c4[3] * (s5 * s5 - s4 * s4);
            dq[4][7] = 2.0 * c4[2] * s3 * s7 + c4[4] * s4 * s5;
        }
    }
    {
        double s0 = S[0], s1 = S[1], s2 = S[2];
        double p = s1 * s1 + s2 * s2;
        out[5] = c5[0] * s0 * s0 * s0 * s0 + c5[1] * s0 * s0 * p + c5[2] * p * p;
        if (dq) {
            dq[5][0] = 4.0 * c5[0] * s0 * s0 * s0 + 2.0 * c5[1] * s0 * p;
            dq[5][1] = 2.0 * c5[1] * s0 * s0 * s1 + 4.0 * c5[2] * p * s1;
            dq[5][2] = 2.0 * c5[1] * s0 * s0 * s2 + 4.0 * c5[2] * p * s2;
        }
    }
}

/* ---- network, Eq. (1) / Listing 1 PAPER.md:912-963 ---------------------------------------------- */
void onep_ann(int D, int H, const double* w0, const double* b0, const double* w1, const double* b1,
              const double* q, double* energy, double* fp)
{
    double e = 0.0;
    for (int d = 0; d < D; ++d) fp[d] = 0.0;
    for (int n = 0; n < H; ++n) {
        double s = 0.0;
        for (int d = 0; d < D; ++d) s += w0[n * D + d] * q[d];
        double x1 = tanh(s - b0[n]);
        double tanh_der = 1.0 - x1 * x1;
        e += w1[n] * x1;
        for (int d = 0; d < D; ++d) fp[d] += w1[n] * (tanh_der * w0[n * D + d]);
    }
    *energy = e - b1[0];
}

/* ---- O1: minimum image + neighbour predicate (readings A8, A8t) -----------------------
 * The cell is box[9] = rows a, b, c (lattice vectors).
 * Orthorhombic cell (all off-diagonal elements zero), reading A8, literally:
 *   each component: d = (r_j - r_i) - L * rint((r_j - r_i)/L) on periodic axes.
 * General (triclinic) cell, reading A8t: t = r_j - r_i; fractional s_k = (t_x Hinv[x][k] + t_y Hinv[y][k])
 *   + t_z Hinv[z][k] with Hinv the inverse of H = box by cofactors; n_k = rint(s_k) on periodic lattice
 *   directions; d = ((t - n_a a) - n_b b) - n_c c.  This is the nearest image whenever |d| is below half the
 *   smallest perpendicular width of the cell, which the harness guarantees for every cutoff it uses.
 * d2 = (dx*dx + dy*dy) + dz*dz in IEEE fp64 without contraction; neighbour iff d2 < rc*rc (strict). */
static void inverse3(const double H[9], double inv[9])
{
    const double c00 = H[4] * H[8] - H[5] * H[7], c01 = H[5] * H[6] - H[3] * H[8], c02 = H[3] * H[7] - H[4] * H[6];
    const double det = (H[0] * c00 + H[1] * c01) + H[2] * c02;
    inv[0] = c00 / det; inv[1] = (H[2] * H[7] - H[1] * H[8]) / det; inv[2] = (H[1] * H[5] - H[2] * H[4]) / det;
    inv[3] = c01 / det; inv[4] = (H[0] * H[8] - H[2] * H[6]) / det; inv[5] = (H[2] * H[3] - H[0] * H[5]) / det;
    inv[6] = c02 / det; inv[7] = (H[1] * H[6] - H[0] * H[7]) / det; inv[8] = (H[0] * H[4] - H[1] * H[3]) / det;
}

static void min_image(const double* ri, const double* rj, const double box[9], const int32_t pbc[3], double d[3])
{
    const int diagonal = box[1] == 0.0 && box[2] == 0.0 && box[3] == 0.0 && box[5] == 0.0 && box[6] == 0.0 && box[7] == 0.0;
    if (diagonal) {
        for (int a = 0; a < 3; ++a) {
            double t = rj[a] - ri[a];
            if (pbc[a]) t = t - box[4 * a] * rint(t / box[4 * a]);
            d[a] = t;
        }
        return;
    }
    double inv[9], t[3], nk[3];
    inverse3(box, inv);
    for (int a = 0; a < 3; ++a) t[a] = rj[a] - ri[a];
    for (int k = 0; k < 3; ++k) {
        const double sk = (t[0] * inv[k] + t[1] * inv[3 + k]) + t[2] * inv[6 + k];    /* row vector times Hinv */
        nk[k] = pbc[k] ? rint(sk) : 0.0;
    }
    for (int a = 0; a < 3; ++a) d[a] = ((t[a] - nk[0] * box[a]) - nk[1] * box[3 + a]) - nk[2] * box[6 + a];
}
static double dist2(const double d[3]) { return (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]; }

/* brute force list: count[i], list[i*cap + m]; entries beyond cap are counted but not stored.
 * returns the largest count (so the caller can detect cap overflow).                               */
int64_t onep_neighbors(int64_t n, const double* pos, const double box[9], const int32_t pbc[3],
                       double rc, int32_t* count, int32_t* list, int64_t cap)
{
    int64_t maxc = 0;
    double rc2 = rc * rc;
#pragma omp parallel for schedule(static) reduction(max : maxc)
    for (int64_t i = 0; i < n; ++i) {
        int64_t c = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double d[3];
            min_image(pos + 3 * i, pos + 3 * j, box, pbc, d);
            if (dist2(d) < rc2) {
                if (c < cap) list[i * cap + c] = (int32_t)j;
                ++c;
            }
        }
        count[i] = (int32_t)c;
        if (c > maxc) maxc = c;
    }
    return maxc;
}

/* neighbours of a chosen subset of atoms only (O(n_sel * N)); used for sampled full-size parity.   */
int64_t onep_neighbors_of(int64_t n, const double* pos, const double box[9], const int32_t pbc[3],
                          double rc, int64_t n_sel, const int64_t* sel, int32_t* count, int32_t* list, int64_t cap)
{
    int64_t maxc = 0;
    double rc2 = rc * rc;
#pragma omp parallel for schedule(static) reduction(max : maxc)
    for (int64_t s = 0; s < n_sel; ++s) {
        int64_t i = sel[s], c = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double d[3];
            min_image(pos + 3 * i, pos + 3 * j, box, pbc, d);
            if (dist2(d) < rc2) {
                if (c < cap) list[s * cap + c] = (int32_t)j;
                ++c;
            }
        }
        count[s] = (int32_t)c;
        if (c > maxc) maxc = c;
    }
    return maxc;
}

/* ---- O2-O6: energy, force, virial ----------------------------------------------------------------
 * Parameter layouts (same as the library's ABI, stated in include/nep.h):
 *   c_radial[T][T][NR][KR] index (t_i, t_j, n, k); c_angular[T][T][NA][KA]; w0[H][D]; b0[H]; w1[H]; b1[1].
 * Descriptor order (reading A2): nu = n for the radial block; then blocks l=1,2,3,4, 4-body, 5-body,
 *   nu = NR + blk*NA + n.
 * Outputs: energy[n], force[n][3], virial[n][9] with W[a][b] = sum_j r_ij^a (dU_j/dr_ji)^b (Eq. 24).
 * Optional (may be NULL): q[n][D], fp[n][D], S[n][NA][24].
 * Returns 0, or -1 on allocation failure.                                                           */
typedef struct { int32_t j; double d[3]; double r; } pair_t;

static pair_t* build_pairs(int64_t n, const double* pos, const double box[9], const int32_t pbc[3],
                           double rc, int64_t** first_out)
{
    int64_t* first = (int64_t*)malloc(sizeof(int64_t) * (size_t)(n + 1));
    int32_t* cnt = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    if (!first || !cnt) { free(first); free(cnt); return NULL; }
    double rc2 = rc * rc;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        int32_t c = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double d[3];
            min_image(pos + 3 * i, pos + 3 * j, box, pbc, d);
            if (dist2(d) < rc2) ++c;
        }
        cnt[i] = c;
    }
    first[0] = 0;
    for (int64_t i = 0; i < n; ++i) first[i + 1] = first[i] + cnt[i];
    pair_t* pairs = (pair_t*)malloc(sizeof(pair_t) * (size_t)(first[n] > 0 ? first[n] : 1));
    if (!pairs) { free(first); free(cnt); return NULL; }
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        int64_t p = first[i];
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double d[3];
            min_image(pos + 3 * i, pos + 3 * j, box, pbc, d);
            double d2 = dist2(d);
            if (d2 < rc2) {
                pairs[p].j = (int32_t)j;
                pairs[p].d[0] = d[0]; pairs[p].d[1] = d[1]; pairs[p].d[2] = d[2];
                pairs[p].r = sqrt(d2);
                ++p;
            }
        }
    }
    free(cnt);
    *first_out = first;
    return pairs;
}

/* Cells of any size (reading A18): the sums of Eqs. (2) and (12) run over ALL atoms of the periodic
 * structure within r_c, i.e. over every lattice image (j, N) with |r_j + N_a a + N_b b + N_c c - r_i| < r_c,
 * (j, N) != (i, 0) -- in a cell thinner than 2 r_c several images of the same j (and images of i itself) count.
 * Plain loop over image shifts: t = r_j - r_i; N0_k = rint((t Hinv)_k); for m in [-M_k, M_k]^3: N = N0 + m,
 * d = ((t - N_a a) - N_b b) - N_c c; neighbour iff (dx dx + dy dy) + dz dz < rc rc (strict), with
 * M_k = floor(rc / width_k + 1/2) + 1 and width_k the distance between the cell faces k.                     */
static pair_t* build_pairs_images(int64_t n, const double* pos, const double box[9], double rc, int64_t** first_out)
{
    double inv[9];
    inverse3(box, inv);
    int M[3];
    for (int k = 0; k < 3; ++k) {
        const double w = 1.0 / sqrt(inv[k] * inv[k] + inv[3 + k] * inv[3 + k] + inv[6 + k] * inv[6 + k]);
        M[k] = (int)floor(rc / w + 0.5) + 1;
    }
    int64_t* first = (int64_t*)malloc(sizeof(int64_t) * (size_t)(n + 1));
    if (!first) return NULL;
    const double rc2 = rc * rc;
    pair_t* pairs = NULL;
    for (int pass = 0; pass < 2; ++pass) {              /* count, then fill */
        int64_t p = 0;
        for (int64_t i = 0; i < n; ++i) {
            if (pass == 0) first[i] = p;
            for (int64_t j = 0; j < n; ++j) {
                double t[3], n0[3];
                for (int a = 0; a < 3; ++a) t[a] = pos[3 * j + a] - pos[3 * i + a];
                for (int k = 0; k < 3; ++k) n0[k] = rint((t[0] * inv[k] + t[1] * inv[3 + k]) + t[2] * inv[6 + k]);
                for (int ma = -M[0]; ma <= M[0]; ++ma)
                    for (int mb = -M[1]; mb <= M[1]; ++mb)
                        for (int mc = -M[2]; mc <= M[2]; ++mc) {
                            const double N[3] = {n0[0] + ma, n0[1] + mb, n0[2] + mc};
                            if (j == i && N[0] == 0.0 && N[1] == 0.0 && N[2] == 0.0) continue;
                            double d[3];
                            for (int a = 0; a < 3; ++a) d[a] = ((t[a] - N[0] * box[a]) - N[1] * box[3 + a]) - N[2] * box[6 + a];
                            const double d2 = dist2(d);
                            if (d2 < rc2) {
                                if (pass == 1) {
                                    pairs[p].j = (int32_t)j;
                                    pairs[p].d[0] = d[0]; pairs[p].d[1] = d[1]; pairs[p].d[2] = d[2];
                                    pairs[p].r = sqrt(d2);
                                }
                                ++p;
                            }
                        }
            }
        }
        if (pass == 0) {
            first[n] = p;
            pairs = (pair_t*)malloc(sizeof(pair_t) * (size_t)(p > 0 ? p : 1));
            if (!pairs) { free(first); return NULL; }
        }
    }
    *first_out = first;
    return pairs;
}

static int compute_impl(const onep_hyper* h,
                 const double* c_radial, const double* c_angular,
                 const double* w0, const double* b0, const double* w1, const double* b1,
                 int64_t n, const double* pos, const int32_t* type, const double box[9], const int32_t pbc[3], int images,
                 double* energy, double* force, double* virial,
                 double* q_out, double* fp_out, double* S_out);

static double g_last_search_s = 0.0, g_last_eval_s = 0.0;    /* see onep_last_timing */
static double wall_seconds(void)
{
#ifdef _OPENMP
    return omp_get_wtime();
#else
    return 0.0;
#endif
}

int onep_compute(const onep_hyper* h,
                 const double* c_radial, const double* c_angular,
                 const double* w0, const double* b0, const double* w1, const double* b1,
                 int64_t n, const double* pos, const int32_t* type, const double box[9], const int32_t pbc[3],
                 double* energy, double* force, double* virial,
                 double* q_out, double* fp_out, double* S_out)
{
    return compute_impl(h, c_radial, c_angular, w0, b0, w1, b1, n, pos, type, box, pbc, 0, energy, force, virial, q_out, fp_out, S_out);
}

/* the same for a fully periodic cell of ANY size: neighbours are all lattice images within the cutoffs
 * (build_pairs_images; reading A18).  Everything after the pair lists is the code of onep_compute.        */
int onep_compute_images(const onep_hyper* h,
                 const double* c_radial, const double* c_angular,
                 const double* w0, const double* b0, const double* w1, const double* b1,
                 int64_t n, const double* pos, const int32_t* type, const double box[9],
                 double* energy, double* force, double* virial,
                 double* q_out, double* fp_out, double* S_out)
{
    const int32_t pbc[3] = {1, 1, 1};
    return compute_impl(h, c_radial, c_angular, w0, b0, w1, b1, n, pos, type, box, pbc, 1, energy, force, virial, q_out, fp_out, S_out);
}

/* number of ordered neighbour entries (j, N) within rc of each atom, lattice images counted (test hook)  */
int onep_count_images(int64_t n, const double* pos, const double box[9], double rc, int32_t* count)
{
    int64_t* first = NULL;
    pair_t* P = build_pairs_images(n, pos, box, rc, &first);
    if (!P) return -1;
    for (int64_t i = 0; i < n; ++i) count[i] = (int32_t)(first[i + 1] - first[i]);
    free(P); free(first);
    return 0;
}

static int compute_impl(const onep_hyper* h,
                 const double* c_radial, const double* c_angular,
                 const double* w0, const double* b0, const double* w1, const double* b1,
                 int64_t n, const double* pos, const int32_t* type, const double box[9], const int32_t pbc[3], int images,
                 double* energy, double* force, double* virial,
                 double* q_out, double* fp_out, double* S_out)
{
    const int T = h->n_types;
    const int NR = h->n_max_radial + 1, KR = h->basis_radial + 1;
    const int NA = h->n_max_angular + 1, KA = h->basis_angular + 1;
    const int D = onep_num_descriptors(h), H = h->n_neurons;
    const int has4 = h->l_max_4b >= 2, has5 = h->l_max_5b >= 1, L3 = h->l_max_3b;
    const int blk4 = L3, blk5 = L3 + has4;        /* block indices of the 4-body and 5-body components */
    int nk_used = 0;                               /* number of S_k needed for l <= l_max_3b */
    for (int k = 0; k < NUM_B; ++k) if (L_OF_K[k] <= L3) nk_used = k + 1;
    if (has4 && nk_used < 8) nk_used = 8;
    if (has5 && nk_used < 3) nk_used = 3;

    int64_t *firstR = NULL, *firstA = NULL;
    const double t_begin = wall_seconds();
    pair_t* PR = images ? build_pairs_images(n, pos, box, h->rc_radial, &firstR) : build_pairs(n, pos, box, pbc, h->rc_radial, &firstR);
    pair_t* PA = images ? build_pairs_images(n, pos, box, h->rc_angular, &firstA) : build_pairs(n, pos, box, pbc, h->rc_angular, &firstA);
    const double t_lists = wall_seconds();
    double* q = (double*)calloc((size_t)(n * D + 1), sizeof(double));
    double* fp = (double*)calloc((size_t)(n * D + 1), sizeof(double));
    double* S = (double*)calloc((size_t)(n * NA * NUM_B + 1), sizeof(double));
    double* pfR = PR ? (double*)calloc((size_t)(3 * firstR[n] + 1), sizeof(double)) : NULL;
    double* pfA = PA ? (double*)calloc((size_t)(3 * firstA[n] + 1), sizeof(double)) : NULL;
    if (!PR || !PA || !q || !fp || !S || !pfR || !pfA) {
        free(PR); free(PA); free(firstR); free(firstA); free(q); free(fp); free(S); free(pfR); free(pfA);
        return -1;
    }

    /* O2, O3, O4: descriptors and network, one atom at a time */
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i) {
        double fk[64];
        double* qi = q + i * D;
        double* Si = S + i * NA * NUM_B;
        const int ti = type[i];
        /* Eq. (2)-(3): q_n = sum_j sum_k c^{ij}_{nk} f_k(r_ij) */
        for (int64_t p = firstR[i]; p < firstR[i + 1]; ++p) {
            const int tj = type[PR[p].j];
            onep_fk(PR[p].r, h->rc_radial, h->basis_radial, fk, NULL);
            for (int nn = 0; nn < NR; ++nn) {
                double g = 0.0;
                for (int k = 0; k < KR; ++k) g += c_radial[((ti * T + tj) * NR + nn) * KR + k] * fk[k];
                qi[nn] += g;
            }
        }
        /* Eq. (12): S_nk = sum_j g_n(r_ij) b_k(r_ij)/r_ij^{l_k}  (own cutoff, basis, coefficients) */
        for (int64_t p = firstA[i]; p < firstA[i + 1]; ++p) {
            const int tj = type[PA[p].j];
            double b[NUM_B];
            onep_fk(PA[p].r, h->rc_angular, h->basis_angular, fk, NULL);
            onep_bk(PA[p].d, b);
            for (int nn = 0; nn < NA; ++nn) {
                double g = 0.0;
                for (int k = 0; k < KA; ++k) g += c_angular[((ti * T + tj) * NA + nn) * KA + k] * fk[k];
                for (int k = 0; k < NUM_B; ++k) Si[nn * NUM_B + k] += g * b[k] / pow(PA[p].r, L_OF_K[k]);
            }
        }
        /* Eqs. (13)-(19) */
        for (int nn = 0; nn < NA; ++nn) {
            double out[6];
            onep_q_from_S(Si + nn * NUM_B, out, NULL);
            for (int l = 1; l <= L3; ++l) qi[NR + (l - 1) * NA + nn] = out[l - 1];
            if (has4) qi[NR + blk4 * NA + nn] = out[4];
            if (has5) qi[NR + blk5 * NA + nn] = out[5];
        }
        /* Eq. (1) */
        onep_ann(D, H, w0, b0, w1, b1, qi, &energy[i], fp + i * D);
    }

    /* O5: partial forces dU_i/dr_ij for every ordered pair, Eq. (21) */
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i) {
        double fk[64], dfk[64];
        const int ti = type[i];
        const double* fpi = fp + i * D;
        const double* Si = S + i * NA * NUM_B;
        /* first term of Eq. (21): sum_n dU/dq_n g_n'(r) r_hat */
        for (int64_t p = firstR[i]; p < firstR[i + 1]; ++p) {
            const int tj = type[PR[p].j];
            const double r = PR[p].r;
            onep_fk(r, h->rc_radial, h->basis_radial, fk, dfk);
            double s = 0.0;
            for (int nn = 0; nn < NR; ++nn) {
                double dg = 0.0;
                for (int k = 0; k < KR; ++k) dg += c_radial[((ti * T + tj) * NR + nn) * KR + k] * dfk[k];
                s += fpi[nn] * dg;
            }
            for (int a = 0; a < 3; ++a) pfR[3 * p + a] = s * PR[p].d[a] / r;
        }
        /* last three terms of Eq. (21): sum_n sum_k G_nk grad[ g_n(r) P_k(r_vec) / r^l ],
         * G_nk = dU_i/dS_nk = sum_blocks dU/dq_block * dq_block/dS_nk                              */
        for (int64_t p = firstA[i]; p < firstA[i + 1]; ++p) {
            const int tj = type[PA[p].j];
            const double r = PA[p].r;
            const double* d = PA[p].d;
            double b[NUM_B], gb[NUM_B][3], acc[3] = {0.0, 0.0, 0.0};
            onep_fk(r, h->rc_angular, h->basis_angular, fk, dfk);
            onep_bk(d, b);
            onep_bk_grad(d, gb);
            for (int nn = 0; nn < NA; ++nn) {
                double g = 0.0, dg = 0.0, out[6], dq[6][NUM_B];
                for (int k = 0; k < KA; ++k) {
                    double c = c_angular[((ti * T + tj) * NA + nn) * KA + k];
                    g += c * fk[k];
                    dg += c * dfk[k];
                }
                onep_q_from_S(Si + nn * NUM_B, out, dq);
                for (int k = 0; k < nk_used; ++k) {
                    const int l = L_OF_K[k];
                    double G = 0.0;
                    if (l <= L3) G += fpi[NR + (l - 1) * NA + nn] * dq[l - 1][k];
                    if (has4) G += fpi[NR + blk4 * NA + nn] * dq[4][k];
                    if (has5) G += fpi[NR + blk5 * NA + nn] * dq[5][k];
                    /* grad[g P_k r^-l] = (g'/r^(l+1) - l g/r^(l+2)) P_k r_vec + g r^-l grad P_k */
                    double radial = dg / pow(r, l + 1) - l * g / pow(r, l + 2);
                    for (int a = 0; a < 3; ++a)
                        acc[a] += G * (radial * b[k] * d[a] + g / pow(r, l) * gb[k][a]);
                }
            }
            for (int a = 0; a < 3; ++a) pfA[3 * p + a] = acc[a];
        }
    }

    /* O6: F_i = sum_j [dU_i/dr_ij - dU_j/dr_ji] (Eqs. 22-23); W_i = sum_j r_ij (x) dU_j/dr_ji (Eq. 24).
     * Evaluated by visiting every ordered pair (i->j) once: its partial force enters F_i with +,
     * F_j with -, and W_j through r_ji = -r_ij.  Serial, so the sums are deterministic.            */
    for (int64_t i = 0; i < 3 * n; ++i) force[i] = 0.0;
    for (int64_t i = 0; i < 9 * n; ++i) virial[i] = 0.0;
    for (int pass = 0; pass < 2; ++pass) {
        const pair_t* P = pass ? PA : PR;
        const int64_t* first = pass ? firstA : firstR;
        const double* pf = pass ? pfA : pfR;
        for (int64_t i = 0; i < n; ++i)
            for (int64_t p = first[i]; p < first[i + 1]; ++p) {
                const int64_t j = P[p].j;
                for (int a = 0; a < 3; ++a) {
                    force[3 * i + a] += pf[3 * p + a];
                    force[3 * j + a] -= pf[3 * p + a];
                    for (int bb = 0; bb < 3; ++bb) virial[9 * j + 3 * a + bb] += (-P[p].d[a]) * pf[3 * p + bb];
                }
            }
    }

    if (q_out) memcpy(q_out, q, sizeof(double) * (size_t)(n * D));
    if (fp_out) memcpy(fp_out, fp, sizeof(double) * (size_t)(n * D));
    if (S_out) memcpy(S_out, S, sizeof(double) * (size_t)(n * NA * NUM_B));
    free(PR); free(PA); free(firstR); free(firstA); free(q); free(fp); free(S); free(pfR); free(pfA);
    g_last_search_s = t_lists - t_begin;
    g_last_eval_s = wall_seconds() - t_lists;
    return 0;
}

/* Wall-clock split of the last onep_compute / onep_compute_images call (bench.py's cpu_baseline: BASELINE.md
 * section 3 wants the evaluation given the lists and the O(N^2) search reported separately):
 * out[0] = seconds in the brute-force pair search, out[1] = seconds in O2-O6.  Timing only; no arithmetic.  */
void onep_last_timing(double out[2]) { out[0] = g_last_search_s; out[1] = g_last_eval_s; }

/* ---- O7: velocity-Verlet NVE -------------------------------------------------------------------
 * per step: v += (dt/2) F/m;  r += dt v;  F = F(r);  v += (dt/2) F/m.   Units: eV, Angstrom, amu, fs:
 * a[Angstrom/fs^2] = F/m * 9.648533212e-3.  Neighbours are brute-forced at the exact cutoffs every
 * step (a skin list changes nothing: f_c vanishes at r_c).  Positions are not wrapped.
 * e_pot[s], e_kin[s] (s = 0..n_steps) receive the energies before the first and after each step.  */
int onep_md(const onep_hyper* h,
            const double* c_radial, const double* c_angular,
            const double* w0, const double* b0, const double* w1, const double* b1,
            int64_t n, double* pos, double* vel, const int32_t* type, const double* mass_amu,
            const double box[9], const int32_t pbc[3], double dt_fs, int32_t n_steps,
            double* e_pot, double* e_kin)
{
    const double conv = 9.648533212e-3;
    double* en = (double*)malloc(sizeof(double) * (size_t)n);
    double* f = (double*)malloc(sizeof(double) * (size_t)(3 * n));
    double* w = (double*)malloc(sizeof(double) * (size_t)(9 * n));
    if (!en || !f || !w) { free(en); free(f); free(w); return -1; }
    int rc = onep_compute(h, c_radial, c_angular, w0, b0, w1, b1, n, pos, type, box, pbc, en, f, w, NULL, NULL, NULL);
    for (int s = 0; s <= n_steps && rc == 0; ++s) {
        double ep = 0.0, ek = 0.0;
        for (int64_t i = 0; i < n; ++i) {
            ep += en[i];
            for (int a = 0; a < 3; ++a) ek += 0.5 * mass_amu[type[i]] * vel[3 * i + a] * vel[3 * i + a] / conv;
        }
        if (e_pot) e_pot[s] = ep;
        if (e_kin) e_kin[s] = ek;
        if (s == n_steps) break;
        for (int64_t i = 0; i < n; ++i)
            for (int a = 0; a < 3; ++a) {
                vel[3 * i + a] += 0.5 * dt_fs * f[3 * i + a] / mass_amu[type[i]] * conv;
                pos[3 * i + a] += dt_fs * vel[3 * i + a];
            }
        rc = onep_compute(h, c_radial, c_angular, w0, b0, w1, b1, n, pos, type, box, pbc, en, f, w, NULL, NULL, NULL);
        for (int64_t i = 0; i < n; ++i)
            for (int a = 0; a < 3; ++a)
                vel[3 * i + a] += 0.5 * dt_fs * f[3 * i + a] / mass_amu[type[i]] * conv;
    }
    free(en); free(f); free(w);
    return rc;
}
