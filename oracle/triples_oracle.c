/*
 * oracle/triples_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU evaluation of the closed-shell CCSD(T) perturbative
 * triples energy E(T) = E[4] + E[5] of arXiv:1609.08094 (section 2.2).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code with the CUDA path.
 *
 * Every function follows the paper's equations literally, in fp64, with direct loops over
 * i,j,k,a,b,c and inner loops over d (virtual) and l (occupied):
 *
 *   Eq. (2.2.2), L94 : t_ijk^abc = -P_ijk^abc [ sum_d t_ij^ad g_ckbd - sum_l t_il^ab g_cklj ] / eps_ijk^abc
 *   Eq. (2.2.3), L99 : P x_ijk^abc = x_ijk^abc + x_ikj^acb + x_jik^bac + x_jki^bca + x_kij^cab + x_kji^cba
 *   Eq. (2.2.4): z_ijk^abc = -( t_i^a g_jbkc + t_j^b g_iakc + t_k^c g_iajb ) / eps_ijk^abc
 *   Eq. (2.2.5): x~^abc   = 2 ( 2/3 x^abc - x^acb + 1/3 x^bca )
 *   Eq. (2.2.1), L87 : E[4] = sum t~ t eps ,  E[5] = sum z~ t eps        (sign: reading Q1 below)
 *   eps_ijk^abc "on par with" Eq. (2.1.2), L65/L92: eps_a + eps_b + eps_c - (eps_i + eps_j + eps_k)
 *
 * Integral classes, Mulliken notation (L63), row-major, last index fastest:
 *   g_ckbd = (ck|bd) = (bd|ck) = vvvo[b][d][c][k]      vvvo[a][b][c][k] = (ab|ck)
 *   g_cklj = (ck|lj)           = ovoo[k][c][l][j]      ovoo[i][a][j][k] = (ia|jk)
 *   g_jbkc = (jb|kc)           = ovov[j][b][k][c]      ovov[i][a][j][b] = (ia|jb)
 *   t2[i][j][a][b] = t_ij^ab,  t1[i][a] = t_i^a
 *
 * Readings of the paper:
 *   Q1  Taken literally, Eq. (2.2.1) with eps = virt - occ > 0 gives +sum W~ V / eps, the
 *       negative of the textbook (T) energy (refs 9, 64 of the paper).  We use
 *       E[4] = -sum t~ t eps, E[5] = -sum z~ t eps, i.e. sum W~ (W+Vd) / D with
 *       D = occ - virt < 0.  tests/test_oracle_pins.py pins this sign against the spin-orbital
 *       textbook formula by brute force.
 *   Q4  Restricted loop i<=j<=k (L119, Eq. (5.0.7b)): the paper gives no weights.  Mode
 *       (ii) uses weight (2 - delta_ij - delta_jk) and the six-term symmetrised combination
 *       Z[W]^abc = 4W^abc + W^bca + W^cab - 2W^acb - 2W^cba - 2W^bac; it is checked against the
 *       literal unrestricted sum (mode (i)) in the tests.
 *
 * Pins: see tests/test_oracle_pins.py (P1..P9 of SURVEY.md 8(c)).  Absolute values of E(T) on
 * the synthetic inputs are "parity unpinned by the paper" (no worked example is printed).
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (oracle/build_oracle.py).  OpenMP is used only the way
 * the paper's CPU code uses it (L121): one composite loop over the independent ijk cycles,
 * each thread with a private W block.
 */
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long long i64;

#define T1(i, a) t1[(i64)(i) * v + (a)]
#define T2(i, j, a, b) t2[(((i64)(i) * o + (j)) * v + (a)) * v + (b)]
#define VVVO(a, b, c, k) vvvo[(((i64)(a) * v + (b)) * v + (c)) * o + (k)]
#define OVOO(i, a, j, k) ovoo[(((i64)(i) * v + (a)) * o + (j)) * o + (k)]
#define OVOV(i, a, j, b) ovov[(((i64)(i) * v + (a)) * o + (j)) * v + (b)]

/* Numerator of Eq. (2.2.2) for one ordered index set before P is applied:
 *   x_pqr^{a'b'c'} = sum_d t_pq^{a'd} g_{c'r b'd} - sum_l t_pl^{a'b'} g_{c'r l q}            */
static double x_term(int o, int v, const double *t2, const double *vvvo, const double *ovoo,
                     int p, int q, int r, int a, int b, int c)
{
    double s = 0.0;
    for (int d = 0; d < v; ++d) s += T2(p, q, a, d) * VVVO(b, d, c, r);   /* (c r | b d) */
    for (int l = 0; l < o; ++l) s -= T2(p, l, a, b) * OVOO(r, c, l, q);   /* (c r | l q) */
    return s;
}

/* W_ijk^abc = P_ijk^abc x_ijk^abc, Eq. (2.2.3): W[(a*v+b)*v+c]. */
static void w_block(int o, int v, const double *t2, const double *vvvo, const double *ovoo,
                    int i, int j, int k, double *W)
{
    for (int a = 0; a < v; ++a)
        for (int b = 0; b < v; ++b)
            for (int c = 0; c < v; ++c)
                W[((i64)a * v + b) * v + c] =
                    x_term(o, v, t2, vvvo, ovoo, i, j, k, a, b, c) +
                    x_term(o, v, t2, vvvo, ovoo, i, k, j, a, c, b) +
                    x_term(o, v, t2, vvvo, ovoo, j, i, k, b, a, c) +
                    x_term(o, v, t2, vvvo, ovoo, j, k, i, b, c, a) +
                    x_term(o, v, t2, vvvo, ovoo, k, i, j, c, a, b) +
                    x_term(o, v, t2, vvvo, ovoo, k, j, i, c, b, a);
}

/* Numerator of Eq. (2.2.4): Vd_ijk^abc = t_i^a g_jbkc + t_j^b g_iakc + t_k^c g_iajb. */
static double vd_term(int o, int v, const double *t1, const double *ovov,
                      int i, int j, int k, int a, int b, int c)
{
    return T1(i, a) * OVOV(j, b, k, c) + T1(j, b) * OVOV(i, a, k, c) + T1(k, c) * OVOV(i, a, j, b);
}

/* Mode (i) cycle: literal Eq. (2.2.1)-(2.2.5) for one ORDERED (i,j,k):
 *   e4 = -sum_abc t~ t eps,  e5 = -sum_abc z~ t eps   (sign: Q1).                            */
static void cycle_literal(int o, int v, const double *eps_o, const double *eps_v, const double *t1,
                          const double *t2, const double *vvvo, const double *ovoo, const double *ovov,
                          int i, int j, int k, double *W, long double *e4, long double *e5)
{
    w_block(o, v, t2, vvvo, ovoo, i, j, k, W);
    long double s4 = 0.0L, s5 = 0.0L;
#define WW(a, b, c) W[((i64)(a) * v + (b)) * v + (c)]
    for (int a = 0; a < v; ++a)
        for (int b = 0; b < v; ++b)
            for (int c = 0; c < v; ++c) {
                double eps = eps_v[a] + eps_v[b] + eps_v[c] - (eps_o[i] + eps_o[j] + eps_o[k]);
                /* eps is symmetric in abc, so the permuted amplitudes share it */
                double t_abc = -WW(a, b, c) / eps;
                double t_acb = -WW(a, c, b) / eps;
                double t_bca = -WW(b, c, a) / eps;
                double z_abc = -vd_term(o, v, t1, ovov, i, j, k, a, b, c) / eps;
                double z_acb = -vd_term(o, v, t1, ovov, i, j, k, a, c, b) / eps;
                double z_bca = -vd_term(o, v, t1, ovov, i, j, k, b, c, a) / eps;
                double tt = 2.0 * (2.0 / 3.0 * t_abc - t_acb + 1.0 / 3.0 * t_bca); /* Eq. (2.2.5) */
                double zt = 2.0 * (2.0 / 3.0 * z_abc - z_acb + 1.0 / 3.0 * z_bca);
                s4 += (long double)(tt * t_abc * eps);
                s5 += (long double)(zt * t_abc * eps);
            }
    *e4 = -s4;
    *e5 = -s5;
}

/* Mode (ii) cycle for one restricted triplet i<=j<=k (reading Q4), unweighted:
 *   e4 = sum_abc Z[W] W / D,  e5 = sum_abc Z[W] Vd / D,  D = occ - virt.                     */
static void cycle_restricted(int o, int v, const double *eps_o, const double *eps_v, const double *t1,
                             const double *t2, const double *vvvo, const double *ovoo, const double *ovov,
                             int i, int j, int k, double *W, long double *e4, long double *e5)
{
    w_block(o, v, t2, vvvo, ovoo, i, j, k, W);
    long double s4 = 0.0L, s5 = 0.0L;
    for (int a = 0; a < v; ++a)
        for (int b = 0; b < v; ++b)
            for (int c = 0; c < v; ++c) {
                double D = eps_o[i] + eps_o[j] + eps_o[k] - eps_v[a] - eps_v[b] - eps_v[c];
                double Z = 4.0 * WW(a, b, c) + WW(b, c, a) + WW(c, a, b)
                         - 2.0 * WW(a, c, b) - 2.0 * WW(c, b, a) - 2.0 * WW(b, a, c);
                s4 += (long double)(Z * WW(a, b, c) / D);
                s5 += (long double)(Z * vd_term(o, v, t1, ovov, i, j, k, a, b, c) / D);
            }
#undef WW
    *e4 = s4;
    *e5 = s5;
}

static int bad_args(int o, int v, const void *p0, const void *p1, const void *p2, const void *p3,
                    const void *p4, const void *p5, const void *p6)
{
    return o < 1 || v < 1 || !p0 || !p1 || !p2 || !p3 || !p4 || !p5 || !p6;
}

/* Mode (i): the literal unrestricted sum over ALL ordered i,j,k (o^3 cycles).
 * out[0] = E(T), out[1] = E[4], out[2] = E[5].  Returns 0 on success.                        */
int oracle_triples_unrestricted(int o, int v, const double *eps_o, const double *eps_v, const double *t1,
                                const double *t2, const double *vvvo, const double *ovoo,
                                const double *ovov, double *out)
{
    if (bad_args(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov) || !out) return 1;
    i64 n = (i64)o * o * o;
    long double *p4 = (long double *)calloc((size_t)n, sizeof(long double));
    long double *p5 = (long double *)calloc((size_t)n, sizeof(long double));
    if (!p4 || !p5) { free(p4); free(p5); return 2; }
    int fail = 0;
#pragma omp parallel
    {
        double *W = (double *)malloc(sizeof(double) * (size_t)v * v * v);
        if (!W) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp for schedule(dynamic)
        for (i64 t = 0; t < n; ++t) {
            if (!W) continue;
            int i = (int)(t / ((i64)o * o)), j = (int)((t / o) % o), k = (int)(t % o);
            cycle_literal(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, i, j, k, W, &p4[t], &p5[t]);
        }
        free(W);
    }
    long double e4 = 0.0L, e5 = 0.0L;
    for (i64 t = 0; t < n; ++t) { e4 += p4[t]; e5 += p5[t]; }   /* fixed order */
    free(p4); free(p5);
    if (fail) return 2;
    out[1] = (double)e4; out[2] = (double)e5; out[0] = (double)(e4 + e5);
    return 0;
}

/* Per-triplet energies for a list of restricted triplets (i<=j<=k required):
 *   e_out[3*n+0] = w*(e4+e5), e_out[3*n+1] = w*e4, e_out[3*n+2] = w*e5, w = 2 - d_ij - d_jk.  */
int oracle_triples_subset(int o, int v, const double *eps_o, const double *eps_v, const double *t1,
                          const double *t2, const double *vvvo, const double *ovoo, const double *ovov,
                          int ntrip, const int *trip, double *e_out)
{
    if (bad_args(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov) || ntrip < 0 || (ntrip && (!trip || !e_out)))
        return 1;
    for (int n = 0; n < ntrip; ++n) {
        int i = trip[3 * n], j = trip[3 * n + 1], k = trip[3 * n + 2];
        if (i < 0 || i > j || j > k || k >= o) return 1;
    }
    int fail = 0;
#pragma omp parallel
    {
        double *W = (double *)malloc(sizeof(double) * (size_t)v * v * v);
        if (!W) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp for schedule(dynamic)
        for (int n = 0; n < ntrip; ++n) {
            if (!W) continue;
            int i = trip[3 * n], j = trip[3 * n + 1], k = trip[3 * n + 2];
            long double e4, e5;
            cycle_restricted(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, i, j, k, W, &e4, &e5);
            double w = 2.0 - (i == j ? 1.0 : 0.0) - (j == k ? 1.0 : 0.0);
            e_out[3 * n + 1] = (double)(w * e4);
            e_out[3 * n + 2] = (double)(w * e5);
            e_out[3 * n + 0] = (double)(w * (e4 + e5));
        }
        free(W);
    }
    return fail ? 2 : 0;
}

/* Mode (ii): restricted sum over i<=j<=k in the enumeration order
 *   for i in [0,o): for j in [i,o): for k in [j,o)       (Eq. (5.0.7b))
 * out[0..2] = E(T), E[4], E[5]; e_triplet (optional, 3*T doubles) as in oracle_triples_subset. */
int oracle_triples_restricted(int o, int v, const double *eps_o, const double *eps_v, const double *t1,
                              const double *t2, const double *vvvo, const double *ovoo, const double *ovov,
                              double *out, double *e_triplet)
{
    if (bad_args(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov) || !out) return 1;
    int T = (int)((i64)o * (o + 1) * (o + 2) / 6);
    int *trip = (int *)malloc(sizeof(int) * 3 * (size_t)T);
    double *e = e_triplet ? e_triplet : (double *)malloc(sizeof(double) * 3 * (size_t)T);
    if (!trip || !e) { free(trip); if (!e_triplet) free(e); return 2; }
    int n = 0;
    for (int i = 0; i < o; ++i)
        for (int j = i; j < o; ++j)
            for (int k = j; k < o; ++k) { trip[3 * n] = i; trip[3 * n + 1] = j; trip[3 * n + 2] = k; ++n; }
    int rc = oracle_triples_subset(o, v, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, T, trip, e);
    if (rc == 0) {
        long double e4 = 0.0L, e5 = 0.0L;
        for (int t = 0; t < T; ++t) { e4 += e[3 * t + 1]; e5 += e[3 * t + 2]; }   /* fixed order */
        out[1] = (double)e4; out[2] = (double)e5; out[0] = (double)(e4 + e5);
    }
    free(trip);
    if (!e_triplet) free(e);
    return rc;
}

/* W block of one ordered (i,j,k) for elementwise checks: W[v^3], Eq. (2.2.3) numerator. */
int oracle_w_block(int o, int v, const double *t2, const double *vvvo, const double *ovoo,
                   int i, int j, int k, double *W)
{
    if (o < 1 || v < 1 || !t2 || !vvvo || !ovoo || !W) return 1;
    if (i < 0 || j < 0 || k < 0 || i >= o || j >= o || k >= o) return 1;
    w_block(o, v, t2, vvvo, ovoo, i, j, k, W);
    return 0;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
