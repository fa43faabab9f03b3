/* Every entry point of oracle/fmm_oracle.c on small seeded inputs, to be built together with it under
 * -fsanitize=address,undefined (tests/test_oracle_sanitize.py).  Exit code 0 = no finding; the
 * sanitizers abort on the first one (-fno-sanitize-recover=all).  Values are checked only for being finite: what
 * they should BE is the business of the pins. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

int fmm_oracle_stencil(double, int, int, int *, signed char *);
int fmm_oracle_stencil_leaf(double, int, int, int *, signed char *);
int fmm_oracle_green(const double *, double *);
int fmm_oracle_pair(const double *, const double *, double, const double *, int, double *, double *);
int fmm_oracle_interact_multipole(const int *, const int *, const int *, double, double, int, const double *, const double *,
                                  double *, double *, unsigned long long *);
int fmm_oracle_interact_multipole_cond(const int *, const int *, const int *, double, double, int, const double *,
                                       const double *, double *, double *, double *, unsigned long long *);
int fmm_oracle_interact_multipole_mixed(const int *, const int *, const int *, double, double, int, const double *,
                                        const double *, const unsigned char *, double *, double *, unsigned long long *);
int fmm_oracle_interact_monopole(const int *, const int *, const int *, double, double, const double *, double *,
                                 unsigned long long *);
int fmm_oracle_interact_monopole_leaf(const int *, const int *, const int *, double, double, const double *, double *,
                                      unsigned long long *);
int fmm_oracle_interaction_count(const int *, const int *, const int *, double, unsigned long long *);
int fmm_oracle_m2m(const int *, double, const double *, const double *, double *, double *);
int fmm_oracle_m2m_about(const int *, double, const double *, const double *, const double *, double *);
int fmm_oracle_l2l(const int *, double, const double *, const double *, const double *, const double *, double *, double *);
int fmm_oracle_direct_sum(const int *, double, const double *, double *);
int fmm_oracle_tree_interact_multipole(const int *, double, double, int, const double *, const double *, const unsigned char *,
                                       double *, double *, unsigned long long *);
int fmm_oracle_tree_leaf_p2p(const int *, double, double, const unsigned char *, const double *, double *, unsigned long long *);
int fmm_oracle_tree_cross_level(const int *, double, double, const unsigned char *, const double *, const unsigned char *,
                                const double *, double *, double *, unsigned long long *);
int fmm_oracle_direct_sum_points(long, const double *, const double *, double *);

static unsigned long long rs = 88172645463325252ULL;
static double u01(void)
{
    rs ^= rs << 13; rs ^= rs >> 7; rs ^= rs << 17;
    return (double)(rs >> 11) * (1.0 / 9007199254740992.0);
}
static int finite_all(const double *a, size_t n)
{
    for (size_t i = 0; i < n; ++i)
        if (!isfinite(a[i])) return 0;
    return 1;
}
#define CHECK(c) do { if (!(c)) { fprintf(stderr, "oracle_sanitize: check failed at line %d\n", __LINE__); return 1; } } while (0)

int main(void)
{
    const double theta[3] = {0.5, 0.35, 0.7};
    for (int t = 0; t < 3; ++t)
        for (int par = 0; par < 8; ++par) {
            int cnt = 0, cnt2 = 0;
            CHECK(fmm_oracle_stencil(theta[t], par, 0, &cnt, NULL) == 0 && cnt > 0);
            signed char *d = (signed char *)malloc((size_t)3 * cnt);
            CHECK(fmm_oracle_stencil(theta[t], par, cnt, &cnt2, d) == 0 && cnt2 == cnt);
            free(d);
            CHECK(fmm_oracle_stencil_leaf(theta[t], par, 0, &cnt2, NULL) == 0 && cnt2 > cnt);
        }
    double R[3] = {3.0, 1.0, 2.0}, G[121], MB[20], MA3[10], Lp[20], dL[3];
    CHECK(fmm_oracle_green(R, G) == 0 && finite_all(G, 121));
    for (int c = 0; c < 20; ++c) MB[c] = u01() - 0.3;
    for (int c = 0; c < 10; ++c) MA3[c] = 0.01 * (u01() - 0.5);
    CHECK(fmm_oracle_pair(R, MB, 1.5, MA3, 1, Lp, dL) == 0 && finite_all(Lp, 20) && finite_all(dL, 3));

    /* a 16 x 8 x 24 level: multipole step (whole grid and a ragged region), condition output, mixed level, monopoles */
    const int n[3] = {16, 8, 24}, lo0[3] = {0, 0, 0}, lo[3] = {3, 1, 5}, hi[3] = {11, 8, 17};
    const size_t nc = (size_t)n[0] * n[1] * n[2];
    const double h = 0.37;
    double *mom = (double *)malloc(20 * nc * 8), *com = (double *)malloc(3 * nc * 8);
    unsigned char *leaf = (unsigned char *)malloc(nc);
    for (size_t i = 0; i < 20 * nc; ++i) mom[i] = (i < nc ? 0.5 + u01() : 0.01 * (u01() - 0.5)) * h * h * h;
    for (size_t i = 0; i < 3 * nc; ++i) com[i] = 0.2 * h * (u01() - 0.5);
    for (size_t i = 0; i < nc; ++i) leaf[i] = (unsigned char)(((i / 8) & 1) != 0);
    double *L = (double *)malloc(20 * nc * 8), *C = (double *)malloc(3 * nc * 8), *A = (double *)malloc(23 * nc * 8);
    unsigned long long cnt = 0, cnt2 = 0;
    for (int t = 0; t < 3; ++t) {
        CHECK(fmm_oracle_interact_multipole(n, lo0, n, h, theta[t], 1, mom, com, L, C, &cnt) == 0 && finite_all(L, 20 * nc));
        CHECK(fmm_oracle_interaction_count(n, lo0, n, theta[t], &cnt2) == 0 && cnt2 == cnt);
        CHECK(fmm_oracle_interact_multipole(n, lo, hi, h, theta[t], 0, mom, com, L, NULL, &cnt) == 0);
        CHECK(fmm_oracle_interact_multipole_cond(n, lo, hi, h, theta[t], 1, mom, com, L, C, A, &cnt) == 0 && finite_all(A, 23 * 8 * 7 * 12));
        CHECK(fmm_oracle_interact_multipole_mixed(n, lo0, n, h, theta[t], 1, mom, com, leaf, L, C, &cnt) == 0 && cnt > cnt2);
        CHECK(fmm_oracle_interact_monopole(n, lo, hi, h, theta[t], mom, L, &cnt) == 0);
        CHECK(fmm_oracle_interact_monopole_leaf(n, lo0, n, h, theta[t], mom, L, &cnt) == 0 && finite_all(L, 4 * nc));
    }
    CHECK(fmm_oracle_direct_sum(n, h, mom, L) == 0 && finite_all(L, 4 * nc));
    /* M2M, M2M about given centres, L2L */
    const size_t pc = nc / 8;
    double *pm = (double *)malloc(20 * pc * 8), *po = (double *)malloc(3 * pc * 8), *pm2 = (double *)malloc(20 * pc * 8);
    CHECK(fmm_oracle_m2m(n, h, mom, com, pm, po) == 0 && finite_all(pm, 20 * pc) && finite_all(po, 3 * pc));
    CHECK(fmm_oracle_m2m_about(n, h, mom, com, po, pm2) == 0 && finite_all(pm2, 20 * pc));
    double *pL = (double *)malloc(20 * pc * 8), *pC = (double *)malloc(3 * pc * 8);
    for (size_t i = 0; i < 20 * pc; ++i) pL[i] = u01() - 0.5;
    for (size_t i = 0; i < 3 * pc; ++i) pC[i] = u01() - 0.5;
    memset(L, 0, 20 * nc * 8);
    memset(C, 0, 3 * nc * 8);
    CHECK(fmm_oracle_l2l(n, h, pL, pC, po, com, L, C) == 0 && finite_all(L, 20 * nc) && finite_all(C, 3 * nc));
    CHECK(fmm_oracle_l2l(n, h, pL, NULL, po, com, L, NULL) == 0);
    /* adaptive tree: a 16^3 coarse level whose low-x half is refined, the 32^3 level below it */
    const int c3[3] = {16, 16, 16}, f3[3] = {32, 32, 32};
    const size_t cc = 4096, fc = 32768;
    unsigned char *kc = (unsigned char *)malloc(cc), *kf = (unsigned char *)malloc(fc);
    double *mc = (double *)malloc(cc * 8), *mf = (double *)malloc(fc * 8);
    for (size_t i = 0; i < cc; ++i) { kc[i] = (i % 16) < 8 ? 2 : 1; mc[i] = kc[i] == 1 ? 0.5 + u01() : 0.0; }
    for (size_t i = 0; i < fc; ++i) { kf[i] = (i % 32) < 16 ? 1 : 0; mf[i] = kf[i] == 1 ? 0.0625 * (0.5 + u01()) : 0.0; }
    double *tm = (double *)calloc(20 * cc, 8), *to = (double *)calloc(3 * cc, 8), *tL = (double *)malloc(20 * cc * 8), *tC = (double *)malloc(3 * cc * 8);
    for (size_t i = 0; i < cc; ++i) tm[i] = 0.5 + u01();
    CHECK(fmm_oracle_tree_interact_multipole(c3, 1.0 / 16, 0.5, 1, tm, to, kc, tL, tC, &cnt) == 0 && finite_all(tL, 20 * cc) && cnt > 0);
    double *oc = (double *)calloc(4 * cc, 8), *of = (double *)calloc(4 * fc, 8);
    CHECK(fmm_oracle_tree_leaf_p2p(c3, 1.0 / 16, 0.5, kc, mc, oc, &cnt) == 0 && cnt > 0);
    CHECK(fmm_oracle_tree_leaf_p2p(f3, 1.0 / 32, 0.35, kf, mf, of, &cnt) == 0 && cnt > 0);
    CHECK(fmm_oracle_tree_cross_level(c3, 1.0 / 16, 0.5, kc, mc, kf, mf, oc, of, &cnt) == 0 && cnt > 0 && finite_all(oc, 4 * cc) && finite_all(of, 4 * fc));
    CHECK(fmm_oracle_tree_cross_level(c3, 1.0 / 16, 0.7, kc, mc, kf, mf, oc, of, &cnt) == 0);
    kf[0] = 2;                                  /* a fine cell that is not a leaf next to a coarse leaf?  (0,0,0) is far from x >= 8: still fine */
    CHECK(fmm_oracle_tree_cross_level(c3, 1.0 / 16, 0.5, kc, mc, kf, mf, oc, of, &cnt) == 0);
    kf[(size_t)15] = 2;                         /* fine cell x = 15: child of the refined cell next to the coarse leaf x = 8: refused */
    CHECK(fmm_oracle_tree_cross_level(c3, 1.0 / 16, 0.5, kc, mc, kf, mf, oc, of, &cnt) != 0);
    double pos[3 * 64], pmass[64], pout[4 * 64];
    for (int i = 0; i < 64; ++i) { pmass[i] = u01(); for (int a = 0; a < 3; ++a) pos[3 * i + a] = u01(); }
    CHECK(fmm_oracle_direct_sum_points(64, pos, pmass, pout) == 0 && finite_all(pout, 256));
    free(mom); free(com); free(leaf); free(L); free(C); free(A); free(pm); free(po); free(pm2); free(pL); free(pC);
    free(kc); free(kf); free(mc); free(mf); free(tm); free(to); free(tL); free(tC); free(oc); free(of);
    printf("oracle_sanitize: ok\n");
    return 0;
}
