/*
 * fmm_oracle.c -- plain, slow, obviously-correct CPU oracle of the same-level FMM
 * cell-to-cell interaction step of Octo-Tiger's gravity solver.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may build, load or call it.  It
 * shares no code, header, table or constant with the CUDA path under
 * paper_2101_08226_b200/ and neither includes the other.
 *
 * What it follows (PAPER.md = arxiv 2101.08226, section 2.2):
 *   - "variant of the Cartesian FMM described by Dehnen (2000) ... conserves linear
 *     momentum to machine precision ... Both multipole and expansions are relative to
 *     cell centres" (L125);
 *   - the angular-momentum extension that "works by adding an additional higher order
 *     multipoles which is used to calculate a correction to the calculated force" while
 *     "preserving linear momentum conservation" (L127);
 *   - the opening criterion, Eq. 15 (L131-135): theta' = dx/|x_A - x_B| < theta  <=>  well
 *     separated; two cells interact here "when they are well separated from each other,
 *     but their respective parents are not well separated";
 *   - isolated boundary: the FMM ignores the domain boundary (L321); G = 1 (L363).
 * The paper prints no FMM formulas (it defers to Dehnen 2000 / Marcello et al. 2016), so
 * the formulas are the readings listed in DESIGN.md ("Readings of the paper") and
 * SURVEY.md section 8(c), restated here step by step with FULL (non-unique) tensors:
 *
 *   Green's function g(R) = -1/|R| and its derivative tensors D^(n) = d^n g / dR^n,
 *     d0=-1/r, d1=1/r^3, d2=-3/r^5, d3=15/r^7, d4=-105/r^9,
 *     D0 = d0;  D1_i = d1 R_i;  D2_ij = d1 d_ij + d2 R_i R_j;
 *     D3_ijk = d2 (d_ij R_k + d_ik R_j + d_jk R_i) + d3 R_i R_j R_k;
 *     D4_ijkl = d2 (d_ij d_kl + d_ik d_jl + d_il d_jk)
 *             + d3 (d_ij R_k R_l + d_ik R_j R_l + d_il R_j R_k + d_jk R_i R_l + d_jl R_i R_k + d_kl R_i R_j)
 *             + d4 R_i R_j R_k R_l.
 *   For target A and every partner B of its stencil (R = z_A - z_B, expansion centres =
 *   centres of mass handed over as offsets delta from the geometric cell centre):
 *     L0       += M_B D0 - M1_B.D1 + 1/2 M2_B:D2 - 1/6 M3_B:.D3
 *     L1_i     += M_B D1_i - M1_B,j D2_ij + 1/2 M2_B,jk D3_ijk
 *     L2_ij    += M_B D2_ij - M1_B,k D3_ijk
 *     L3_ijk   += M_B D3_ijk                                   (truncation n + m <= 3)
 *     correction (L127):  n3 = M3_B - (M_B/M_A) M3_A ;  dL1_i += -1/6 n3_jkl D4_ijkl
 *   Monopole (leaf) variant: R = geometric centre difference,
 *     phi += -m_B/|R| ;  g_i += -m_B R_i/|R|^3.
 *
 * Precision: every per-pair term is formed in IEEE double; the running sums over the
 * partners are `long double` (x87 80-bit on this host) so the oracle's own summation
 * error stays out of the 1e-12 parity budget.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): stencil counts and theta_min
 * (L137), worked example W1, symbolic derivatives of -1/r (sympy), order-of-convergence
 * against direct summation over point masses, Newton's third law (L125), angular-momentum
 * conservation with the correction on and its violation with it off (L127), point-mass
 * and uniform-sphere closed forms; for the passes of the complete solve (M2M, M2M about prescribed
 * centres, L2L, leaf list, direct sum; tests/test_oracle_solve.py): P2M of all constituents, the symbolic
 * Taylor shift, the exact point sum, conservation, the uniform-sphere residuals of Table 1, and for the
 * second right-hand side (L81-83) proportionality to the density's solve and linearity.
 * No function here is "parity unpinned".
 *
 * Layouts: moments [20][nz][ny][nx] (monopole: [1][nz][ny][nx]), com_off [3][nz][ny][nx],
 * outputs SoA over the output region: L [20][oz][oy][ox], Lcorr [3][oz][oy][ox],
 * monopole out [4][oz][oy][ox] = (phi, gx, gy, gz).  x is the fastest index.
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_EINVAL 1
#define ORC_EMASS 2

/* ---------------------------------------------------------------------------------- */
/* Opening criterion, Eq. 15 (L131-135).  Distances are in units of the cell width, so  */
/* theta' = 1/|Delta|;  "theta' < theta"  <=>  |Delta|^2 theta^2 > 1  (strict, L135).   */
/* ---------------------------------------------------------------------------------- */
static int well_separated(long d2, double theta) { return (double)d2 * theta * theta > 1.0; }

/* parent index of a cell index: floor(i/2), also for negative i */
static int parent_of(int i) { return (i >= 0) ? (i / 2) : -((-i + 1) / 2); }

/* Is Delta a partner of a cell with parity (px,py,pz)?  Cells well separated (L135),      */
/* parents not well separated; a parent is never well separated from itself (Delta_I = 0). */
/* leaf != 0: the leaf-level list of the complete solve (NEXT f1) -- every Delta != 0 whose parents are not */
/* well separated, i.e. the Eq. 15 list plus the near field (cells that are not well separated, L135/L456). */
static int is_partner_mode(int px, int py, int pz, int dx, int dy, int dz, double theta, int leaf)
{
    long d2 = (long)dx * dx + (long)dy * dy + (long)dz * dz;
    if (d2 == 0 || (!leaf && !well_separated(d2, theta))) return 0;
    int Ix = parent_of(px + dx) - parent_of(px);
    int Iy = parent_of(py + dy) - parent_of(py);
    int Iz = parent_of(pz + dz) - parent_of(pz);
    long D2 = (long)Ix * Ix + (long)Iy * Iy + (long)Iz * Iz;
    if (D2 > 0 && well_separated(D2, theta)) return 0;
    return 1;
}

/* search range that certainly contains the stencil: parents within 1/theta parent cells */
static int search_reach(double theta) { return 2 * (int)floor(1.0 / theta) + 3; }

/* Stencil of parity class parity = px + 2 py + 4 pz, in lexicographic (dz, dy, dx) order. */
/* dxyz receives up to cap triples (dx,dy,dz); *count is always the full count.           */
static int stencil_mode(double theta, int parity, int leaf, int cap, int *count, signed char *dxyz)
{
    if (!(theta > 0.0 && theta < 1.0) || parity < 0 || parity > 7 || !count) return ORC_EINVAL;
    int px = parity & 1, py = (parity >> 1) & 1, pz = (parity >> 2) & 1;
    int S = search_reach(theta), c = 0;
    if (S > 127) return ORC_EINVAL;
    for (int dz = -S; dz <= S; ++dz)
        for (int dy = -S; dy <= S; ++dy)
            for (int dx = -S; dx <= S; ++dx)
                if (is_partner_mode(px, py, pz, dx, dy, dz, theta, leaf)) {
                    if (dxyz && c < cap) {
                        dxyz[3 * c + 0] = (signed char)dx;
                        dxyz[3 * c + 1] = (signed char)dy;
                        dxyz[3 * c + 2] = (signed char)dz;
                    }
                    ++c;
                }
    *count = c;
    return ORC_OK;
}
int fmm_oracle_stencil(double theta, int parity, int cap, int *count, signed char *dxyz)
{
    return stencil_mode(theta, parity, 0, cap, count, dxyz);
}
/* leaf-level list of the complete solve: Eq. 15 list + near field (see is_partner_mode) */
int fmm_oracle_stencil_leaf(double theta, int parity, int cap, int *count, signed char *dxyz)
{
    return stencil_mode(theta, parity, 1, cap, count, dxyz);
}

/* ---------------------------------------------------------------------------------- */
/* unique <-> full tensors, lexicographic unique order                                   */
/* ---------------------------------------------------------------------------------- */
static void sort3(int *a, int *b, int *c)
{
    int t;
    if (*a > *b) { t = *a; *a = *b; *b = t; }
    if (*b > *c) { t = *b; *b = *c; *c = t; }
    if (*a > *b) { t = *a; *a = *b; *b = t; }
}
/* position of sorted (i<=j) in [xx xy xz yy yz zz] */
static int u2(int i, int j)
{
    if (i > j) { int t = i; i = j; j = t; }
    static const int tab[3][3] = {{0, 1, 2}, {-1, 3, 4}, {-1, -1, 5}};
    return tab[i][j];
}
/* position of sorted (i<=j<=k) in [xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz] */
static int u3(int i, int j, int k)
{
    sort3(&i, &j, &k);
    static const int tab[3][3][3] = {
        {{0, 1, 2}, {-1, 3, 4}, {-1, -1, 5}},
        {{-1, -1, -1}, {-1, 6, 7}, {-1, -1, 8}},
        {{-1, -1, -1}, {-1, -1, -1}, {-1, -1, 9}}};
    return tab[i][j][k];
}

static double kd(int i, int j) { return i == j ? 1.0 : 0.0; }

/* Green's-function derivative tensors of g = -1/|R| (closed forms in the header).       */
static void green_tensors(const double R[3], double *D0, double D1[3], double D2[3][3],
                          double D3[3][3][3], double D4[3][3][3][3])
{
    double r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
    double r = sqrt(r2);
    double d0 = -1.0 / r;
    double d1 = 1.0 / (r2 * r);
    double d2 = -3.0 / (r2 * r2 * r);
    double d3 = 15.0 / (r2 * r2 * r2 * r);
    double d4 = -105.0 / (r2 * r2 * r2 * r2 * r);
    *D0 = d0;
    for (int i = 0; i < 3; ++i) {
        D1[i] = d1 * R[i];
        for (int j = 0; j < 3; ++j) {
            D2[i][j] = d1 * kd(i, j) + d2 * R[i] * R[j];
            for (int k = 0; k < 3; ++k) {
                D3[i][j][k] = d2 * (kd(i, j) * R[k] + kd(i, k) * R[j] + kd(j, k) * R[i]) + d3 * R[i] * R[j] * R[k];
                if (D4)
                    for (int l = 0; l < 3; ++l)
                        D4[i][j][k][l] =
                            d2 * (kd(i, j) * kd(k, l) + kd(i, k) * kd(j, l) + kd(i, l) * kd(j, k)) +
                            d3 * (kd(i, j) * R[k] * R[l] + kd(i, k) * R[j] * R[l] + kd(i, l) * R[j] * R[k] +
                                  kd(j, k) * R[i] * R[l] + kd(j, l) * R[i] * R[k] + kd(k, l) * R[i] * R[j]) +
                            d4 * R[i] * R[j] * R[k] * R[l];
            }
        }
    }
}

/* flattened export of the tensors for the symbolic-derivative pin: 1+3+9+27+81 = 121 */
int fmm_oracle_green(const double R[3], double out[121])
{
    double D0, D1[3], D2[3][3], D3[3][3][3], D4[3][3][3][3];
    if (!R || !out) return ORC_EINVAL;
    green_tensors(R, &D0, D1, D2, D3, D4);
    out[0] = D0;
    memcpy(out + 1, D1, sizeof D1);
    memcpy(out + 4, D2, sizeof D2);
    memcpy(out + 13, D3, sizeof D3);
    memcpy(out + 40, D4, sizeof D4);
    return ORC_OK;
}

/* One ordered pair A <- B.  MB = 20 unique source moments; MA0, MA3 = target mass and    */
/* unique third moments (used by the correction only).  term[20] and cterm[3] receive     */
/* this pair's contribution, formed in double.                                            */
static void pair_terms(const double R[3], const double MB[20], double MA0, const double MA3[10],
                       int correction, double term[20], double cterm[3])
{
    double D0, D1[3], D2[3][3], D3[3][3][3], D4[3][3][3][3];
    green_tensors(R, &D0, D1, D2, D3, correction ? D4 : NULL);

    double M0 = MB[0], M1[3], M2[3][3], M3[3][3][3];
    for (int i = 0; i < 3; ++i) {
        M1[i] = MB[1 + i];
        for (int j = 0; j < 3; ++j) {
            M2[i][j] = MB[4 + u2(i, j)];
            for (int k = 0; k < 3; ++k) M3[i][j][k] = MB[10 + u3(i, j, k)];
        }
    }

    /* L0 += M D0 - M1.D1 + 1/2 M2:D2 - 1/6 M3:.D3 */
    double s1 = 0.0, s2 = 0.0, s3 = 0.0;
    for (int i = 0; i < 3; ++i) {
        s1 += M1[i] * D1[i];
        for (int j = 0; j < 3; ++j) {
            s2 += M2[i][j] * D2[i][j];
            for (int k = 0; k < 3; ++k) s3 += M3[i][j][k] * D3[i][j][k];
        }
    }
    term[0] = M0 * D0 - s1 + 0.5 * s2 - s3 / 6.0;

    /* L1_i += M D1_i - M1_j D2_ij + 1/2 M2_jk D3_ijk */
    for (int i = 0; i < 3; ++i) {
        double a = 0.0, b = 0.0;
        for (int j = 0; j < 3; ++j) {
            a += M1[j] * D2[i][j];
            for (int k = 0; k < 3; ++k) b += M2[j][k] * D3[i][j][k];
        }
        term[1 + i] = M0 * D1[i] - a + 0.5 * b;
    }

    /* L2_ij += M D2_ij - M1_k D3_ijk   (unique components i <= j) */
    for (int i = 0; i < 3; ++i)
        for (int j = i; j < 3; ++j) {
            double a = 0.0;
            for (int k = 0; k < 3; ++k) a += M1[k] * D3[i][j][k];
            term[4 + u2(i, j)] = M0 * D2[i][j] - a;
        }

    /* L3_ijk += M D3_ijk   (unique components i <= j <= k) */
    for (int i = 0; i < 3; ++i)
        for (int j = i; j < 3; ++j)
            for (int k = j; k < 3; ++k) term[10 + u3(i, j, k)] = M0 * D3[i][j][k];

    /* correction (L127):  n3 = M3_B - (M_B/M_A) M3_A ;  dL1_i += -1/6 n3_jkl D4_ijkl */
    cterm[0] = cterm[1] = cterm[2] = 0.0;
    if (correction) {
        double q = M0 / MA0;
        for (int i = 0; i < 3; ++i) {
            double c = 0.0;
            for (int j = 0; j < 3; ++j)
                for (int k = 0; k < 3; ++k)
                    for (int l = 0; l < 3; ++l) {
                        double n3 = M3[j][k][l] - q * MA3[u3(j, k, l)];
                        c += n3 * D4[i][j][k][l];
                    }
            cterm[i] = -c / 6.0;
        }
    }
}

/* single ordered pair, for the worked example W1 and closed-form pins */
int fmm_oracle_pair(const double R[3], const double MB[20], double MA0, const double MA3[10],
                    int correction, double L[20], double dL1[3])
{
    if (!R || !MB || !L || !dL1) return ORC_EINVAL;
    if (correction && (!MA3 || !(MA0 > 0.0))) return ORC_EMASS;
    pair_terms(R, MB, MA0, MA3, correction, L, dL1);
    return ORC_OK;
}

static int check_region(const int n[3], const int lo[3], const int hi[3])
{
    for (int a = 0; a < 3; ++a)
        if (n[a] <= 0 || lo[a] < 0 || hi[a] > n[a] || lo[a] >= hi[a]) return 0;
    return 1;
}

/* Build the 8 per-parity partner lists once. */
typedef struct { int count[8]; signed char *d[8]; } stencil_set;

static int build_stencils_mode(double theta, int leaf, stencil_set *S)
{
    memset(S, 0, sizeof *S);
    for (int p = 0; p < 8; ++p) {
        int c = 0;
        if (stencil_mode(theta, p, leaf, 0, &c, NULL) != ORC_OK) return ORC_EINVAL;
        S->d[p] = (signed char *)malloc((size_t)3 * (c > 0 ? c : 1));
        if (!S->d[p]) return ORC_EINVAL;
        stencil_mode(theta, p, leaf, c, &S->count[p], S->d[p]);
    }
    return ORC_OK;
}
static int build_stencils(double theta, stencil_set *S) { return build_stencils_mode(theta, 0, S); }
static void free_stencils(stencil_set *S) { for (int p = 0; p < 8; ++p) free(S->d[p]); }

/*
 * The interaction step for multipole cells.
 * For every target cell A in [out_lo, out_hi): loop over its parity class's partner list
 * in the fixed (dz,dy,dx) order, skip partners outside the grid (isolated, L321),
 * R_c = (double)(i_A,c - i_B,c) * h + (delta_A,c - delta_B,c), accumulate.
 * L gets the correction folded into L1 when enabled; Lcorr (may be NULL) gets it alone.
 * n_interactions (may be NULL) receives the number of ordered in-domain pairs.
 */
enum { TREE_ABSENT = 0, TREE_LEAF = 1, TREE_REFINED = 2 };   /* kind of a cell on one level of an adaptive tree */

static int interact_multipole_impl(const int n[3], const int out_lo[3], const int out_hi[3], double h,
                                   double theta, int am_correction, const double *moments,
                                   const double *com_off, const unsigned char *leaf, const unsigned char *kind,
                                   double *L, double *Lcorr,
                                   double *Labs, unsigned long long *n_interactions)
{
    if (!n || !out_lo || !out_hi || !moments || !com_off || !L || !(h > 0.0)) return ORC_EINVAL;
    if (!check_region(n, out_lo, out_hi)) return ORC_EINVAL;
    stencil_set S;
    /* leaf != NULL (a level of an adaptive mesh, see fmm_oracle_interact_multipole_mixed): candidates are the Eq. 15
     * list plus the near field; a near-field pair counts only if A or B is a leaf cell */
    if (build_stencils_mode(theta, leaf != NULL, &S) != ORC_OK) return ORC_EINVAL;

    const size_t nx = n[0], ny = n[1], nz = n[2], ncell = nx * ny * nz;
    const size_t ox = out_hi[0] - out_lo[0], oy = out_hi[1] - out_lo[1], oz = out_hi[2] - out_lo[2];
    const size_t ocell = ox * oy * oz;
    unsigned long long total = 0;
    int bad_mass = 0;

#pragma omp parallel for collapse(2) schedule(dynamic, 1) reduction(+ : total) reduction(| : bad_mass)
    for (int k = out_lo[2]; k < out_hi[2]; ++k)
        for (int j = out_lo[1]; j < out_hi[1]; ++j)
            for (int i = out_lo[0]; i < out_hi[0]; ++i) {
                const size_t a = ((size_t)k * ny + j) * nx + i;
                const int p = (i & 1) + 2 * (j & 1) + 4 * (k & 1);
                long double acc[20], cacc[3] = {0.0L, 0.0L, 0.0L};
                long double aabs[23];      /* sum over the partners of |term|: the condition of each sum (Labs) */
                for (int c = 0; c < 20; ++c) acc[c] = 0.0L;
                for (int c = 0; c < 23; ++c) aabs[c] = 0.0L;
                double MA3[10], MA0 = moments[a], dA[3];
                for (int c = 0; c < 10; ++c) MA3[c] = moments[(size_t)(10 + c) * ncell + a];
                for (int c = 0; c < 3; ++c) dA[c] = com_off[(size_t)c * ncell + a];
                const int absent = kind && kind[a] == TREE_ABSENT;     /* adaptive tree: no such cell on this level */
                if (am_correction && !(MA0 > 0.0) && !absent) bad_mass |= 1;

                for (int s = 0; s < S.count[p] && !absent; ++s) {
                    const int dx = S.d[p][3 * s], dy = S.d[p][3 * s + 1], dz = S.d[p][3 * s + 2];
                    const int bi = i + dx, bj = j + dy, bk = k + dz;
                    if (bi < 0 || bj < 0 || bk < 0 || bi >= (int)nx || bj >= (int)ny || bk >= (int)nz) continue;
                    const size_t b = ((size_t)bk * ny + bj) * nx + bi;
                    if (leaf && !leaf[a] && !leaf[b] && !is_partner_mode(i & 1, j & 1, k & 1, dx, dy, dz, theta, 0)) continue;
                    /* adaptive tree (fmm_oracle_tree_interact_multipole): B must exist, and two leaf cells meet as point
                     * masses in fmm_oracle_tree_leaf_p2p instead */
                    if (kind && (kind[b] == TREE_ABSENT || (kind[a] == TREE_LEAF && kind[b] == TREE_LEAF))) continue;
                    double MB[20], R[3], term[20], cterm[3];
                    for (int c = 0; c < 20; ++c) MB[c] = moments[(size_t)c * ncell + b];
                    R[0] = (double)(i - bi) * h + (dA[0] - com_off[0 * ncell + b]);
                    R[1] = (double)(j - bj) * h + (dA[1] - com_off[1 * ncell + b]);
                    R[2] = (double)(k - bk) * h + (dA[2] - com_off[2 * ncell + b]);
                    pair_terms(R, MB, MA0, MA3, am_correction && MA0 > 0.0, term, cterm);
                    for (int c = 0; c < 20; ++c) acc[c] += (long double)term[c];
                    for (int c = 0; c < 3; ++c) cacc[c] += (long double)cterm[c];
                    if (Labs) {
                        for (int c = 0; c < 20; ++c) aabs[c] += (long double)fabs(term[c]);
                        for (int c = 0; c < 3; ++c) aabs[20 + c] += (long double)fabs(cterm[c]);
                    }
                    ++total;
                }
                const size_t o = ((size_t)(k - out_lo[2]) * oy + (j - out_lo[1])) * ox + (i - out_lo[0]);
                if (am_correction)
                    for (int c = 0; c < 3; ++c) acc[1 + c] += cacc[c];
                for (int c = 0; c < 20; ++c) L[(size_t)c * ocell + o] = (double)acc[c];
                if (Lcorr)
                    for (int c = 0; c < 3; ++c) Lcorr[(size_t)c * ocell + o] = (double)cacc[c];
                if (Labs)
                    for (int c = 0; c < 23; ++c) Labs[(size_t)c * ocell + o] = (double)aabs[c];
            }
    free_stencils(&S);
    if (n_interactions) *n_interactions = total;
    return bad_mass ? ORC_EMASS : ORC_OK;
}

int fmm_oracle_interact_multipole(const int n[3], const int out_lo[3], const int out_hi[3], double h,
                                  double theta, int am_correction, const double *moments,
                                  const double *com_off, double *L, double *Lcorr,
                                  unsigned long long *n_interactions)
{
    return interact_multipole_impl(n, out_lo, out_hi, h, theta, am_correction, moments, com_off, NULL, NULL, L, Lcorr, NULL, n_interactions);
}

/*
 * The same step, and beside every sum its CONDITION: Labs [23][oz][oy][ox] = sum over the partners of |term| for
 * the 20 coefficients (without the correction) and for the 3 components of the correction.  Nothing of the result
 * depends on it; the parity tests use it to hold each expansion order to 1e-12 of the size of what was summed
 * ("each order normalised by that order's sum_B |term| (condition-aware)") -- in a smooth field the
 * partners' contributions to L2 and to the correction cancel to a small remainder, and an error of n eps sum|term| is
 * then a large fraction of the remainder although every term is right to the last bit.
 */
int fmm_oracle_interact_multipole_cond(const int n[3], const int out_lo[3], const int out_hi[3], double h,
                                       double theta, int am_correction, const double *moments,
                                       const double *com_off, double *L, double *Lcorr, double *Labs,
                                       unsigned long long *n_interactions)
{
    if (!Labs) return ORC_EINVAL;
    return interact_multipole_impl(n, out_lo, out_hi, h, theta, am_correction, moments, com_off, NULL, NULL, L, Lcorr, Labs, n_interactions);
}

/*
 * One level of an ADAPTIVE mesh (a node "is either fully refined with eight child
 * nodes (an interior node) or not refined at all (a leaf node)"; the paper does not describe the gravity side of a
 * refinement boundary -- DESIGN.md reading R8).  leaf[cell] = 1: the cell belongs to a leaf sub-grid (it has no
 * children), 0: to a refined one.  Well-separated pairs (Eq. 15 list) interact here whatever their kind.  A pair that is
 * NOT well separated is normally left to the children (L135); when A or B has none, nobody below will take it, so it is
 * taken here, with the same pair formula (a leaf is the special case M1 = M2 = M3 = 0, delta = 0 of its moments).
 * Hence: partners of A = Eq. 15 list + those near-field cells B for which leaf[A] or leaf[B].
 */
int fmm_oracle_interact_multipole_mixed(const int n[3], const int out_lo[3], const int out_hi[3], double h,
                                        double theta, int am_correction, const double *moments,
                                        const double *com_off, const unsigned char *leaf, double *L, double *Lcorr,
                                        unsigned long long *n_interactions)
{
    if (!leaf) return ORC_EINVAL;
    return interact_multipole_impl(n, out_lo, out_hi, h, theta, am_correction, moments, com_off, leaf, NULL, L, Lcorr, NULL, n_interactions);
}

/*
 * Monopole (leaf) variant (BASELINE.json config 4): every cell is the
 * point mass m at its geometric centre; the same stencil; G = 1 (L363):
 *   phi_A = -sum_B m_B/|R| ,  g_A = -sum_B m_B R/|R|^3 ,  R = x_A - x_B = (i_A - i_B) h.
 * out = [4][oz][oy][ox] = (phi, gx, gy, gz).
 */
static int interact_monopole_mode(const int n[3], const int out_lo[3], const int out_hi[3], double h,
                                  double theta, int leaf, const unsigned char *kind, const double *mass, double *out,
                                  unsigned long long *n_interactions)
{
    if (!n || !out_lo || !out_hi || !mass || !out || !(h > 0.0)) return ORC_EINVAL;
    if (!check_region(n, out_lo, out_hi)) return ORC_EINVAL;
    stencil_set S;
    if (build_stencils_mode(theta, leaf, &S) != ORC_OK) return ORC_EINVAL;
    const size_t nx = n[0], ny = n[1], nz = n[2];
    const size_t ox = out_hi[0] - out_lo[0], oy = out_hi[1] - out_lo[1], oz = out_hi[2] - out_lo[2];
    const size_t ocell = ox * oy * oz;
    unsigned long long total = 0;

#pragma omp parallel for collapse(2) schedule(dynamic, 1) reduction(+ : total)
    for (int k = out_lo[2]; k < out_hi[2]; ++k)
        for (int j = out_lo[1]; j < out_hi[1]; ++j)
            for (int i = out_lo[0]; i < out_hi[0]; ++i) {
                const int p = (i & 1) + 2 * (j & 1) + 4 * (k & 1);
                long double acc[4] = {0.0L, 0.0L, 0.0L, 0.0L};
                /* adaptive tree (fmm_oracle_tree_leaf_p2p): only leaf cells are point masses, as targets and as sources */
                const int skip = kind && kind[((size_t)k * ny + j) * nx + i] != TREE_LEAF;
                for (int s = 0; s < S.count[p] && !skip; ++s) {
                    const int bi = i + S.d[p][3 * s], bj = j + S.d[p][3 * s + 1], bk = k + S.d[p][3 * s + 2];
                    if (bi < 0 || bj < 0 || bk < 0 || bi >= (int)nx || bj >= (int)ny || bk >= (int)nz) continue;
                    if (kind && kind[((size_t)bk * ny + bj) * nx + bi] != TREE_LEAF) continue;
                    const double m = mass[((size_t)bk * ny + bj) * nx + bi];
                    double R[3] = {(double)(i - bi) * h, (double)(j - bj) * h, (double)(k - bk) * h};
                    double r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
                    double r = sqrt(r2);
                    acc[0] += (long double)(-m / r);
                    for (int c = 0; c < 3; ++c) acc[1 + c] += (long double)(-m * R[c] / (r2 * r));
                    ++total;
                }
                const size_t o = ((size_t)(k - out_lo[2]) * oy + (j - out_lo[1])) * ox + (i - out_lo[0]);
                for (int c = 0; c < 4; ++c) out[(size_t)c * ocell + o] = (double)acc[c];
            }
    free_stencils(&S);
    if (n_interactions) *n_interactions = total;
    return ORC_OK;
}

int fmm_oracle_interact_monopole(const int n[3], const int out_lo[3], const int out_hi[3], double h,
                                 double theta, const double *mass, double *out,
                                 unsigned long long *n_interactions)
{
    return interact_monopole_mode(n, out_lo, out_hi, h, theta, 0, NULL, mass, out, n_interactions);
}
/* the same sum over the leaf-level list of the complete solve (Eq. 15 list + near field) */
int fmm_oracle_interact_monopole_leaf(const int n[3], const int out_lo[3], const int out_hi[3], double h,
                                      double theta, const double *mass, double *out,
                                      unsigned long long *n_interactions)
{
    return interact_monopole_mode(n, out_lo, out_hi, h, theta, 1, NULL, mass, out, n_interactions);
}

/* Number of ordered in-domain pairs for a region, by enumeration on the index grid. */
int fmm_oracle_interaction_count(const int n[3], const int out_lo[3], const int out_hi[3], double theta,
                                 unsigned long long *count)
{
    if (!n || !out_lo || !out_hi || !count || !check_region(n, out_lo, out_hi)) return ORC_EINVAL;
    stencil_set S;
    if (build_stencils(theta, &S) != ORC_OK) return ORC_EINVAL;
    unsigned long long total = 0;
#pragma omp parallel for collapse(2) reduction(+ : total)
    for (int k = out_lo[2]; k < out_hi[2]; ++k)
        for (int j = out_lo[1]; j < out_hi[1]; ++j)
            for (int i = out_lo[0]; i < out_hi[0]; ++i) {
                const int p = (i & 1) + 2 * (j & 1) + 4 * (k & 1);
                for (int s = 0; s < S.count[p]; ++s) {
                    const int bi = i + S.d[p][3 * s], bj = j + S.d[p][3 * s + 1], bk = k + S.d[p][3 * s + 2];
                    if (bi < 0 || bj < 0 || bk < 0 || bi >= n[0] || bj >= n[1] || bk >= n[2]) continue;
                    ++total;
                }
            }
    free_stencils(&S);
    *count = total;
    return ORC_OK;
}

int fmm_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void fmm_oracle_set_num_threads(int t)
{
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

/* ====================================================================================== */
/* NEXT f1: the other passes of a complete uniform-grid solve, plain forms.   */
/* "the multipoles of each cell are composed of the multipoles of its child cells ... The   */
/* expansion of each cell is composed of the expansion due to its interactions with other   */
/* cells at the same level, and the expansion of its parent cell".          */
/* Positions are kept RELATIVE to the parent's geometric centre (no O(1) coordinates).      */
/* ====================================================================================== */

/* unique (lexicographic) -> full tensors of one cell */
static void unpack_moments(const double *u, size_t stride, double *M0, double M1[3], double M2[3][3], double M3[3][3][3])
{
    *M0 = u[0];
    for (int i = 0; i < 3; ++i) M1[i] = u[(size_t)(1 + i) * stride];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) M2[i][j] = u[(size_t)(4 + u2(i, j)) * stride];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            for (int k = 0; k < 3; ++k) M3[i][j][k] = u[(size_t)(10 + u3(i, j, k)) * stride];
}

/*
 * M2M: parent multipoles (order 3, about the parent's centre of mass) from its 8 children.
 * nc = child grid (even dims), hc = child cell width; child c of parent P=(I,J,K) is (2I+a,2J+b,2K+c).
 * Child expansion centre relative to the parent's geometric centre: rel = ((a,b,c) - 1/2) hc + delta_c.
 * Parent centre of mass: delta_P = sum_c (M_c rel_c + M1_c) / sum_c M_c   (geometric centre if the mass is 0).
 * Shift of raw moments from z_c to z_P, d = z_c - z_P:
 *   M1'_i = M1_i + M d_i;  M2'_ij = M2_ij + M1_i d_j + M1_j d_i + M d_i d_j;
 *   M3'_ijk = M3_ijk + M2_ij d_k + M2_ik d_j + M2_jk d_i + M1_i d_j d_k + M1_j d_i d_k + M1_k d_i d_j + M d_i d_j d_k.
 * pm = [20][nz/2][ny/2][nx/2], poff = [3][...].
 * given != 0 (second right-hand side, L81-83: the time derivative of the density expanded about the centres
 * of the density itself): delta_P is READ from poff instead of being computed; the shift is the same.
 */
static int m2m_impl(const int nc[3], double hc, const double *cm, const double *coff, double *pm, double *poff, int given)
{
    if (!nc || !cm || !coff || !pm || !poff || !(hc > 0.0)) return ORC_EINVAL;
    for (int a = 0; a < 3; ++a)
        if (nc[a] <= 0 || (nc[a] & 1)) return ORC_EINVAL;
    const size_t cx = nc[0], cy = nc[1], cz = nc[2], ccell = cx * cy * cz;
    const size_t px = cx / 2, py = cy / 2, pz = cz / 2, pcell = px * py * pz;
#pragma omp parallel for collapse(2) schedule(static)
    for (size_t K = 0; K < pz; ++K)
        for (size_t J = 0; J < py; ++J)
            for (size_t I = 0; I < px; ++I) {
                double M0[8], M1[8][3], M2[8][3][3], M3[8][3][3][3], rel[8][3];
                long double mass = 0.0L, com[3] = {0.0L, 0.0L, 0.0L};
                for (int c = 0; c < 8; ++c) {
                    const int a[3] = {c & 1, (c >> 1) & 1, (c >> 2) & 1};
                    const size_t cell = ((2 * K + a[2]) * cy + (2 * J + a[1])) * cx + (2 * I + a[0]);
                    unpack_moments(cm + cell, ccell, &M0[c], M1[c], M2[c], M3[c]);
                    for (int i = 0; i < 3; ++i) rel[c][i] = ((double)a[i] - 0.5) * hc + coff[(size_t)i * ccell + cell];
                    mass += (long double)M0[c];
                    for (int i = 0; i < 3; ++i) com[i] += (long double)(M0[c] * rel[c][i]) + (long double)M1[c][i];
                }
                double dP[3] = {0.0, 0.0, 0.0};
                const size_t P = (K * py + J) * px + I;
                if (given)
                    for (int i = 0; i < 3; ++i) dP[i] = poff[(size_t)i * pcell + P];
                else if (mass != 0.0L)
                    for (int i = 0; i < 3; ++i) dP[i] = (double)(com[i] / mass);
                long double S1[3] = {0, 0, 0}, S2[3][3], S3[3][3][3];
                memset(S2, 0, sizeof S2);
                memset(S3, 0, sizeof S3);
                for (int c = 0; c < 8; ++c) {
                    double d[3];
                    for (int i = 0; i < 3; ++i) d[i] = rel[c][i] - dP[i];
                    for (int i = 0; i < 3; ++i) S1[i] += (long double)(M1[c][i] + M0[c] * d[i]);
                    for (int i = 0; i < 3; ++i)
                        for (int j = 0; j < 3; ++j)
                            S2[i][j] += (long double)(M2[c][i][j] + M1[c][i] * d[j] + M1[c][j] * d[i] + M0[c] * d[i] * d[j]);
                    for (int i = 0; i < 3; ++i)
                        for (int j = 0; j < 3; ++j)
                            for (int k = 0; k < 3; ++k)
                                S3[i][j][k] += (long double)(M3[c][i][j][k] + M2[c][i][j] * d[k] + M2[c][i][k] * d[j] +
                                                             M2[c][j][k] * d[i] + M1[c][i] * d[j] * d[k] + M1[c][j] * d[i] * d[k] +
                                                             M1[c][k] * d[i] * d[j] + M0[c] * d[i] * d[j] * d[k]);
                }
                pm[P] = (double)mass;
                for (int i = 0; i < 3; ++i) pm[(size_t)(1 + i) * pcell + P] = (double)S1[i];
                for (int i = 0; i < 3; ++i)
                    for (int j = i; j < 3; ++j) pm[(size_t)(4 + u2(i, j)) * pcell + P] = (double)S2[i][j];
                for (int i = 0; i < 3; ++i)
                    for (int j = i; j < 3; ++j)
                        for (int k = j; k < 3; ++k) pm[(size_t)(10 + u3(i, j, k)) * pcell + P] = (double)S3[i][j][k];
                if (!given)
                    for (int i = 0; i < 3; ++i) poff[(size_t)i * pcell + P] = dP[i];
            }
    return ORC_OK;
}

int fmm_oracle_m2m(const int nc[3], double hc, const double *cm, const double *coff, double *pm, double *poff)
{
    return m2m_impl(nc, hc, cm, coff, pm, poff, 0);
}

/* M2M about PRESCRIBED parent centres: poff (in) = delta_P of every parent cell; pm (out). */
int fmm_oracle_m2m_about(const int nc[3], double hc, const double *cm, const double *coff, const double *poff, double *pm)
{
    return m2m_impl(nc, hc, cm, coff, pm, (double *)poff, 1);
}

/*
 * L2L: add the parent's local expansion, shifted to the child's expansion centre, to the child's (L125).
 * e = z_c - z_P = ((a,b,c) - 1/2) hc + delta_c - delta_P  (relative to the parent's geometric centre);
 * Taylor shift to order 3:
 *   L0_c += L0 + L1_i e_i + 1/2 L2_ij e_i e_j + 1/6 L3_ijk e_i e_j e_k
 *   L1_c,i += L1_i + L2_ij e_j + 1/2 L3_ijk e_j e_k ;  L2_c,ij += L2_ij + L3_ijk e_k ;  L3_c += L3.
 * The angular-momentum correction is a uniform acceleration of the parent cell and is handed down
 * unchanged: corr_c += corr_P  (pcorr / ccorr may be NULL).
 * pL = [20][parent grid], poff = [3][parent grid], coff = [3][child grid], cL = [20][child grid] (in/out).
 */
int fmm_oracle_l2l(const int nc[3], double hc, const double *pL, const double *pcorr, const double *poff,
                   const double *coff, double *cL, double *ccorr)
{
    if (!nc || !pL || !poff || !coff || !cL || !(hc > 0.0)) return ORC_EINVAL;
    for (int a = 0; a < 3; ++a)
        if (nc[a] <= 0 || (nc[a] & 1)) return ORC_EINVAL;
    const size_t cx = nc[0], cy = nc[1], cz = nc[2], ccell = cx * cy * cz;
    const size_t px = cx / 2, py = cy / 2, pcell = px * py * (cz / 2);
#pragma omp parallel for collapse(2) schedule(static)
    for (size_t k = 0; k < cz; ++k)
        for (size_t j = 0; j < cy; ++j)
            for (size_t i = 0; i < cx; ++i) {
                const size_t cell = (k * cy + j) * cx + i;
                const size_t P = ((k / 2) * py + (j / 2)) * px + (i / 2);
                const int a[3] = {(int)(i & 1), (int)(j & 1), (int)(k & 1)};
                double e[3], L0, L1[3], L2[3][3], L3[3][3][3];
                for (int c = 0; c < 3; ++c)
                    e[c] = ((double)a[c] - 0.5) * hc + coff[(size_t)c * ccell + cell] - poff[(size_t)c * pcell + P];
                unpack_moments(pL + P, pcell, &L0, L1, L2, L3);
                long double s0 = (long double)L0;
                for (int x = 0; x < 3; ++x) {
                    s0 += (long double)(L1[x] * e[x]);
                    for (int y = 0; y < 3; ++y) {
                        s0 += (long double)(0.5 * L2[x][y] * e[x] * e[y]);
                        for (int z = 0; z < 3; ++z) s0 += (long double)(L3[x][y][z] * e[x] * e[y] * e[z] / 6.0);
                    }
                }
                cL[cell] += (double)s0;
                for (int x = 0; x < 3; ++x) {
                    long double s1 = (long double)L1[x];
                    for (int y = 0; y < 3; ++y) {
                        s1 += (long double)(L2[x][y] * e[y]);
                        for (int z = 0; z < 3; ++z) s1 += (long double)(0.5 * L3[x][y][z] * e[y] * e[z]);
                    }
                    cL[(size_t)(1 + x) * ccell + cell] += (double)s1;
                }
                for (int x = 0; x < 3; ++x)
                    for (int y = x; y < 3; ++y) {
                        long double s2 = (long double)L2[x][y];
                        for (int z = 0; z < 3; ++z) s2 += (long double)(L3[x][y][z] * e[z]);
                        cL[(size_t)(4 + u2(x, y)) * ccell + cell] += (double)s2;
                    }
                for (int x = 0; x < 3; ++x)
                    for (int y = x; y < 3; ++y)
                        for (int z = y; z < 3; ++z) cL[(size_t)(10 + u3(x, y, z)) * ccell + cell] += L3[x][y][z];
                if (pcorr && ccorr)
                    for (int c = 0; c < 3; ++c) ccorr[(size_t)c * ccell + cell] += pcorr[(size_t)c * pcell + P];
            }
    return ORC_OK;
}

/*
 * Plain direct sum over point masses on the cell centres of an n^3-type grid (the exact result the
 * complete solve approximates): phi_A = -sum_{B != A} m_B/|R|, g_A = -sum m_B R/|R|^3, G = 1 (L363).
 * out = [4][nz][ny][nx].  O(N^2): for the pins on small grids only.
 */
int fmm_oracle_direct_sum(const int n[3], double h, const double *mass, double *out)
{
    if (!n || !mass || !out || !(h > 0.0)) return ORC_EINVAL;
    const long nx = n[0], ny = n[1], nz = n[2], nc = nx * ny * nz;
#pragma omp parallel for schedule(dynamic, 64)
    for (long a = 0; a < nc; ++a) {
        const long ai = a % nx, aj = (a / nx) % ny, ak = a / (nx * ny);
        long double acc[4] = {0.0L, 0.0L, 0.0L, 0.0L};
        for (long b = 0; b < nc; ++b) {
            if (b == a) continue;
            const long bi = b % nx, bj = (b / nx) % ny, bk = b / (nx * ny);
            const double R[3] = {(double)(ai - bi) * h, (double)(aj - bj) * h, (double)(ak - bk) * h};
            const double r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2], r = sqrt(r2), m = mass[b];
            acc[0] += (long double)(-m / r);
            for (int c = 0; c < 3; ++c) acc[1 + c] += (long double)(-m * R[c] / (r2 * r));
        }
        for (int c = 0; c < 4; ++c) out[(size_t)c * nc + a] = (double)acc[c];
    }
    return ORC_OK;
}


/* ====================================================================================== */
/* NEXT f3: the gravity solve on an ADAPTIVE oct-tree of 8^3 sub-grids.       */
/* PAPER.md L125 ("The FMM adapts naturally to an oct-tree based adaptive mesh refinement"),*/
/* L287-291 (a node "is either fully refined with eight child nodes (an interior node) or   */
/* not refined at all (a leaf node)"; the mesh is properly nested, so a refinement boundary */
/* involves exactly two levels).  The paper does not describe the gravity side of such a    */
/* boundary; reading R9 takes the rule the paper does give (L135: well-separated  */
/* cells interact at the level where their parents are not well separated; what is not well */
/* separated is left to the children, L456) and applies it as a symmetric dual descent:      */
/*   pair (A, B) of one level whose parents are not well separated --                        */
/*     well separated            : they interact here, with the general pair formula; a leaf */
/*                                 is the point mass M0 = m, M1 = M2 = M3 = 0, delta = 0     */
/*                                 (two leaves: that formula IS the point-mass sum, and it   */
/*                                 is taken as such in fmm_oracle_tree_leaf_p2p);            */
/*     not, both refined         : left to their children;                                   */
/*     not, both leaves          : point masses, directly (fmm_oracle_tree_leaf_p2p);        */
/*     not, A leaf and B refined : A meets the eight CHILDREN of B, which proper nesting     */
/*                                 makes leaves one level down: point masses, directly, in   */
/*                                 both directions (fmm_oracle_tree_cross_level).            */
/* Every pair is taken exactly once in each direction with antisymmetric forces, so linear   */
/* momentum -- and with the correction angular momentum -- is conserved as on a uniform grid */
/* (L125, L127), and a fully refined tree is the uniform solve, term by term.                */
/* A level is a dense n^3 array with kind[cell] = TREE_ABSENT / TREE_LEAF / TREE_REFINED.    */
/* ====================================================================================== */

/* the same-level multipole step on one level of the tree: targets = cells that exist; partners = cells of the Eq. 15
 * list that exist, except that two leaves do not meet here.  L (correction folded in) and Lcorr as in
 * fmm_oracle_interact_multipole; absent targets get zeros. */
int fmm_oracle_tree_interact_multipole(const int n[3], double h, double theta, int am_correction,
                                       const double *moments, const double *com_off, const unsigned char *kind,
                                       double *L, double *Lcorr, unsigned long long *n_interactions)
{
    if (!kind) return ORC_EINVAL;
    const int lo[3] = {0, 0, 0};
    return interact_multipole_impl(n, lo, n, h, theta, am_correction, moments, com_off, NULL, kind, L, Lcorr, NULL, n_interactions);
}

/* point-mass sum of the leaf cells of one level over the leaf-level list (Eq. 15 list + near field): targets and sources
 * are the cells with kind == TREE_LEAF.  out = [4][nz][ny][nx] = (phi, g); other targets get zeros. */
int fmm_oracle_tree_leaf_p2p(const int n[3], double h, double theta, const unsigned char *kind, const double *mass,
                             double *out, unsigned long long *n_interactions)
{
    if (!kind) return ORC_EINVAL;
    const int lo[3] = {0, 0, 0};
    return interact_monopole_mode(n, lo, n, h, theta, 1, kind, mass, out, n_interactions);
}

/*
 * The pairs across a refinement boundary.  Coarse level: nc^3-type grid of width hc with kind_c, mass_c; fine level:
 * (2 nc)-type grid of width hc / 2 with kind_f, mass_f.  For every coarse LEAF A and every cell B of its near field (the
 * leaf-level list minus the Eq. 15 list: not well separated, parents not well separated either) that is REFINED, A and
 * each of the 8 children b of B are point masses at their geometric centres:
 *   x_A - x_b = ((double)(2 i_A - i_b) + 0.5) * (hc / 2)      per axis, in this operation order,
 *   out_c[A] += (-m_b / r, -m_b R / r^3),    out_f[b] += (-m_A / r, +m_A R / r^3)   (R = x_A - x_b).
 * A child that is not a leaf means the tree is not properly nested: ORC_EINVAL.  Both outputs are ADDED to
 * ([4][...], long double sums per target in list order, then child order).  n_pairs counts ordered pairs.
 */
int fmm_oracle_tree_cross_level(const int nc[3], double hc, double theta, const unsigned char *kind_c, const double *mass_c,
                                const unsigned char *kind_f, const double *mass_f, double *out_c, double *out_f,
                                unsigned long long *n_pairs)
{
    if (!nc || !kind_c || !mass_c || !kind_f || !mass_f || !out_c || !out_f || !(hc > 0.0)) return ORC_EINVAL;
    stencil_set S;
    if (build_stencils_mode(theta, 1, &S) != ORC_OK) return ORC_EINVAL;
    const long cx = nc[0], cy = nc[1], cz = nc[2], ccell = cx * cy * cz;
    const long fx = 2 * cx, fy = 2 * cy, fz = 2 * cz, fcell = fx * fy * fz;
    const double hf = 0.5 * hc;
    unsigned long long total = 0;
    int bad = 0;
    /* coarse leaf targets */
#pragma omp parallel for collapse(2) schedule(dynamic, 1) reduction(+ : total) reduction(| : bad)
    for (long k = 0; k < cz; ++k)
        for (long j = 0; j < cy; ++j)
            for (long i = 0; i < cx; ++i) {
                const long a = (k * cy + j) * cx + i;
                if (kind_c[a] != TREE_LEAF) continue;
                const int p = (int)((i & 1) + 2 * (j & 1) + 4 * (k & 1));
                long double acc[4] = {0.0L, 0.0L, 0.0L, 0.0L};
                for (int s = 0; s < S.count[p]; ++s) {
                    const int dx = S.d[p][3 * s], dy = S.d[p][3 * s + 1], dz = S.d[p][3 * s + 2];
                    if (well_separated((long)dx * dx + (long)dy * dy + (long)dz * dz, theta)) continue;   /* Eq. 15 list: same level */
                    const long bi = i + dx, bj = j + dy, bk = k + dz;
                    if (bi < 0 || bj < 0 || bk < 0 || bi >= cx || bj >= cy || bk >= cz) continue;
                    if (kind_c[(bk * cy + bj) * cx + bi] != TREE_REFINED) continue;
                    for (int c = 0; c < 8; ++c) {
                        const long ci = 2 * bi + (c & 1), cj = 2 * bj + ((c >> 1) & 1), ck = 2 * bk + (c >> 2);
                        const long b = (ck * fy + cj) * fx + ci;
                        if (kind_f[b] != TREE_LEAF) { bad |= 1; continue; }
                        const double R[3] = {((double)(2 * i - ci) + 0.5) * hf, ((double)(2 * j - cj) + 0.5) * hf,
                                             ((double)(2 * k - ck) + 0.5) * hf};
                        const double r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2], r = sqrt(r2), m = mass_f[b];
                        acc[0] += (long double)(-m / r);
                        for (int x = 0; x < 3; ++x) acc[1 + x] += (long double)(-m * R[x] / (r2 * r));
                        ++total;
                    }
                }
                for (int x = 0; x < 4; ++x) out_c[(long)x * ccell + a] += (double)acc[x];
            }
    /* fine leaf targets: the coarse leaves in the near field of their (refined) parent */
#pragma omp parallel for collapse(2) schedule(dynamic, 1) reduction(+ : total)
    for (long k = 0; k < fz; ++k)
        for (long j = 0; j < fy; ++j)
            for (long i = 0; i < fx; ++i) {
                const long b = (k * fy + j) * fx + i;
                if (kind_f[b] != TREE_LEAF) continue;
                const long pi = i / 2, pj = j / 2, pk = k / 2;
                const int p = (int)((pi & 1) + 2 * (pj & 1) + 4 * (pk & 1));
                long double acc[4] = {0.0L, 0.0L, 0.0L, 0.0L};
                for (int s = 0; s < S.count[p]; ++s) {
                    const int dx = S.d[p][3 * s], dy = S.d[p][3 * s + 1], dz = S.d[p][3 * s + 2];
                    if (well_separated((long)dx * dx + (long)dy * dy + (long)dz * dz, theta)) continue;
                    const long ai = pi + dx, aj = pj + dy, ak = pk + dz;
                    if (ai < 0 || aj < 0 || ak < 0 || ai >= cx || aj >= cy || ak >= cz) continue;
                    const long a = (ak * cy + aj) * cx + ai;
                    if (kind_c[a] != TREE_LEAF) continue;
                    /* R = x_b - x_A = -(x_A - x_b), the latter formed as above */
                    const double R[3] = {-(((double)(2 * ai - i) + 0.5) * hf), -(((double)(2 * aj - j) + 0.5) * hf),
                                         -(((double)(2 * ak - k) + 0.5) * hf)};
                    const double r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2], r = sqrt(r2), m = mass_c[a];
                    acc[0] += (long double)(-m / r);
                    for (int x = 0; x < 3; ++x) acc[1 + x] += (long double)(-m * R[x] / (r2 * r));
                    ++total;
                }
                for (int x = 0; x < 4; ++x) out_f[(long)x * fcell + b] += (double)acc[x];
            }
    free_stencils(&S);
    if (n_pairs) *n_pairs = total;
    return bad ? ORC_EINVAL : ORC_OK;
}

/*
 * Exact sum over point masses at arbitrary positions (the leaves of a tree, whatever their level):
 * phi_a = -sum_{b != a} m_b / |x_a - x_b|,  g_a = -sum m_b (x_a - x_b) / |x_a - x_b|^3.  pos = [np][3], out = [np][4].
 * O(N^2): the exact result the tree solve approximates, for the pins.
 */
int fmm_oracle_direct_sum_points(long np, const double *pos, const double *mass, double *out)
{
    if (np < 0 || !pos || !mass || !out) return ORC_EINVAL;
#pragma omp parallel for schedule(dynamic, 64)
    for (long a = 0; a < np; ++a) {
        long double acc[4] = {0.0L, 0.0L, 0.0L, 0.0L};
        for (long b = 0; b < np; ++b) {
            if (b == a) continue;
            const double R[3] = {pos[3 * a] - pos[3 * b], pos[3 * a + 1] - pos[3 * b + 1], pos[3 * a + 2] - pos[3 * b + 2]};
            const double r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2], r = sqrt(r2);
            acc[0] += (long double)(-mass[b] / r);
            for (int x = 0; x < 3; ++x) acc[1 + x] += (long double)(-mass[b] * R[x] / (r2 * r));
        }
        for (int x = 0; x < 4; ++x) out[4 * a + x] = (double)acc[x];
    }
    return ORC_OK;
}

/* ====================================================================================== */
/* The five calls of the boundary on HOST pointers, under this file's own     */
/* prefix, so that one harness can drive the oracle and the library alike:                  */
/*   fmm_oracle_create / set_moments / interact / get_expansions / destroy.                 */
/* Thin state around the functions above: set_moments copies the caller's arrays, interact  */
/* calls fmm_oracle_interact_multipole or fmm_oracle_interact_monopole on the copy.         */
/* ====================================================================================== */
typedef struct {
    int n[3];
    int out_lo[3], out_hi[3];   /* all zero: the whole grid */
    double h, theta;
    int kind;                   /* 0 multipole, 1 monopole */
    int am_correction;
} fmm_oracle_config;

typedef struct fmm_oracle_handle {
    fmm_oracle_config cfg;
    int lo[3], hi[3];
    size_t ncell, ocell;
    double *mom, *com, *L, *C;
    unsigned long long count;
    int state;                  /* 0 created, 1 sources set, 2 interacted */
} fmm_oracle_t;

int fmm_oracle_destroy(fmm_oracle_t *o)
{
    if (!o) return ORC_EINVAL;
    free(o->mom); free(o->com); free(o->L); free(o->C);
    free(o);
    return ORC_OK;
}

int fmm_oracle_create(const fmm_oracle_config *cfg, fmm_oracle_t **out)
{
    if (!cfg || !out) return ORC_EINVAL;
    *out = NULL;
    if (cfg->kind != 0 && cfg->kind != 1) return ORC_EINVAL;
    if (!(cfg->h > 0.0) || !(cfg->theta > 1.0 / 3.0 && cfg->theta < 1.0)) return ORC_EINVAL;
    fmm_oracle_t *o = (fmm_oracle_t *)calloc(1, sizeof *o);
    if (!o) return ORC_EINVAL;
    o->cfg = *cfg;
    int whole = 1;
    for (int a = 0; a < 3; ++a) whole = whole && cfg->out_lo[a] == 0 && cfg->out_hi[a] == 0;
    for (int a = 0; a < 3; ++a) {
        o->lo[a] = whole ? 0 : cfg->out_lo[a];
        o->hi[a] = whole ? cfg->n[a] : cfg->out_hi[a];
    }
    if (!check_region(cfg->n, o->lo, o->hi)) { free(o); return ORC_EINVAL; }
    o->ncell = (size_t)cfg->n[0] * cfg->n[1] * cfg->n[2];
    o->ocell = (size_t)(o->hi[0] - o->lo[0]) * (o->hi[1] - o->lo[1]) * (o->hi[2] - o->lo[2]);
    const size_t nm = cfg->kind == 0 ? 20 : 1, nl = cfg->kind == 0 ? 20 : 4;
    o->mom = (double *)malloc(nm * o->ncell * sizeof(double));
    o->com = (double *)calloc(3 * o->ncell, sizeof(double));
    o->L = (double *)malloc(nl * o->ocell * sizeof(double));
    o->C = (double *)calloc(3 * o->ocell, sizeof(double));
    if (!o->mom || !o->com || !o->L || !o->C) { fmm_oracle_destroy(o); return ORC_EINVAL; }
    *out = o;
    return ORC_OK;
}

int fmm_oracle_set_moments(fmm_oracle_t *o, const double *moments, const double *com_off)
{
    if (!o || !moments) return ORC_EINVAL;
    memcpy(o->mom, moments, (o->cfg.kind == 0 ? 20 : 1) * o->ncell * sizeof(double));
    if (com_off) memcpy(o->com, com_off, 3 * o->ncell * sizeof(double));
    else memset(o->com, 0, 3 * o->ncell * sizeof(double));
    o->state = 1;
    return ORC_OK;
}

int fmm_oracle_interact(fmm_oracle_t *o)
{
    if (!o) return ORC_EINVAL;
    if (o->state < 1) return ORC_EMASS + 1;        /* "state" error, distinct from EINVAL / EMASS */
    int rc;
    if (o->cfg.kind == 0)
        rc = fmm_oracle_interact_multipole(o->cfg.n, o->lo, o->hi, o->cfg.h, o->cfg.theta, o->cfg.am_correction, o->mom, o->com,
                                           o->L, o->C, &o->count);
    else
        rc = fmm_oracle_interact_monopole(o->cfg.n, o->lo, o->hi, o->cfg.h, o->cfg.theta, o->mom, o->L, &o->count);
    if (rc == ORC_OK || rc == ORC_EMASS) o->state = 2;
    return rc;
}

int fmm_oracle_get_expansions(fmm_oracle_t *o, double *L, double *Lcorr)
{
    if (!o || !L) return ORC_EINVAL;
    if (o->state < 2) return ORC_EMASS + 1;
    memcpy(L, o->L, (o->cfg.kind == 0 ? 20 : 4) * o->ocell * sizeof(double));
    if (Lcorr) {
        if (o->cfg.kind != 0) return ORC_EINVAL;
        memcpy(Lcorr, o->C, 3 * o->ocell * sizeof(double));
    }
    return ORC_OK;
}

int fmm_oracle_handle_interaction_count(const fmm_oracle_t *o, unsigned long long *n)
{
    if (!o || !n || o->state < 2) return ORC_EINVAL;
    *n = o->count;
    return ORC_OK;
}
