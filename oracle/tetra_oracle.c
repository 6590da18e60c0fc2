/*
 * tetra_oracle.c -- plain fp64 CPU oracle for the linear tetrahedron method
 * (orbital-resolved density of states and integrated density of states).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
 * code, header, table or constant with the CUDA path under paper_1710_10789_b200/.
 *
 * What it computes (Eq. 4, :52; Eq. 8-9, :91-97; Eq. 2-3, :43-48):
 *     DOS_m(w) = sum_{tetra i, band n} sum_{l=1..4} b_{n,l,m} dw_{n,l}/dE (w)
 *     N_m(w)   = sum_{tetra i, band n} sum_{l=1..4} b_{n,l,m}  w_{n,l}(w)
 * with the corner weights w_{n,l}(E) of PAPER.md Eq. 11-15 (:105-200), every cube of
 * the periodic N1 x N2 x N3 grid split into the six tetrahedra of Table I (:228-237),
 * the 4 corner energies of each (tetrahedron, band) sorted ascending (:99) and the
 * orbital weight b taken at the matching corner (:243).
 *
 * It follows the paper step by step in the paper's order and notation; every energy
 * point is evaluated for every (tetrahedron, band) exactly as Kernel 3 does (:220),
 * i.e. no windowing, unless `windowed` is requested (see oracle_tetra_dos).
 *
 * Readings of the paper where it is garbled / silent (SURVEY.md
 * 8(c) G1-G17) -- each is exercised by a pin in tests/test_oracle_pins.py:
 *   G1  Eq. 12d: last bracket is (1/E21 + 1/E31 + 1/E41)          (printed 1/E21 twice)
 *   G2  Eq. 12f: denominators are E_j1                            (printed E_i1)
 *   G3  Eq. 13k: w3 = (C1+C2)(E-E1)/E31 + (C2+C3)(E-E2)/E32       (printed E21, E22)
 *   G4  Eq. 13l: last term is (C2+C3)/E32                         (printed C1+C3)
 *   G5  Eq. 14e/f: "(E4 - e)" means (E4 - E)
 *   G7  corner label c=1..8 <-> offset (dx,dy,dz) = bits 0,1,2 of (c-1)
 *   G8  the grid is periodic: N1*N2*N3 cubes, index N_d wraps to 0
 *   G9  V_T/V_G = 1/(6 N1 N2 N3)
 *   G10 half-open intervals, tests in the order E<=E1, E<E2, E<E3, E<E4, else
 *   G11 no special-casing of degenerate corners: an interval of zero length is never
 *       entered, so no vanishing denominator is ever used
 *   G13 f = Theta(w - E_n(k)): states below w are counted
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): derivative consistency,
 * continuity, truncated-power closed form, Monte-Carlo barycentric integration, exact
 * moments, sum rules, closed-form simple-cubic DOS, brute force on tiny grids,
 * invariances.  No function here is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o liboracle.so tetra_oracle.c -lm
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_AOS 0 /* E[ik][n],  W[ik][n][m]  */
#define ORACLE_SOA 1 /* E[n][ik],  W[n][m][ik]  */

/* Table I: corner labels m1..m4 of tetrahedron i = 1..6. */
static const int TABLE_I[6][4] = {
    {1, 2, 3, 6}, {2, 3, 4, 6}, {1, 3, 5, 6}, {3, 4, 6, 8}, {3, 5, 6, 7}, {3, 6, 7, 8}};

int oracle_version(void) { return 1; }

/* Copy of Table I for the geometry pins (6 tetrahedra x 4 labels). */
void oracle_table_I(int out[24]) {
    for (int i = 0; i < 6; i++)
        for (int j = 0; j < 4; j++) out[4 * i + j] = TABLE_I[i][j];
}

/* Reading G7: label c (1..8) -> offset (dx,dy,dz). */
void oracle_corner_offset(int c, int d[3]) {
    d[0] = (c - 1) & 1;
    d[1] = ((c - 1) >> 1) & 1;
    d[2] = ((c - 1) >> 2) & 1;
}

/* Sort 4 energies ascending, keeping the permutation.
 * perm[l] = position in the input of the l-th smallest.  Stable insertion sort. */
void oracle_sort4(const double e_in[4], double e[4], int perm[4]) {
    for (int l = 0; l < 4; l++) {
        e[l] = e_in[l];
        perm[l] = l;
    }
    for (int i = 1; i < 4; i++) {
        double x = e[i];
        int p = perm[i];
        int j = i - 1;
        while (j >= 0 && e[j] > x) {
            e[j + 1] = e[j];
            perm[j + 1] = perm[j];
            j--;
        }
        e[j + 1] = x;
        perm[j + 1] = p;
    }
}

/*
 * Corner weights w_j(E) and derivatives dw_j/dE, j = 1..4, for sorted corner energies
 * e[0] <= e[1] <= e[2] <= e[3] (E1..E4 of PAPER.md:99), V = V_T/(4 V_G).
 * PAPER.md Eq. 10-15 (:101-200) with readings G1-G5, G10, G11.
 * Returns the case: 0 (Eq. 11), 1 (Eq. 12), 2 (Eq. 13), 3 (Eq. 14), 4 (Eq. 15).
 */
int oracle_corner_weights(const double e[4], double E, double V, double w[4], double dw[4]) {
    const double E1 = e[0], E2 = e[1], E3 = e[2], E4 = e[3];
    /* Eq. 10: E_ij = E_i - E_j */
    const double E21 = E2 - E1, E31 = E3 - E1, E41 = E4 - E1;
    const double E32 = E3 - E2, E42 = E4 - E2, E43 = E4 - E3;

    if (E <= E1) { /* Eq. 11 */
        for (int j = 0; j < 4; j++) w[j] = dw[j] = 0.0;
        return 0;
    }
    if (E < E2) { /* Eq. 12a-f */
        const double x = E - E1;
        const double C = V * x * x * x / (E21 * E31 * E41);         /* 12a */
        const double dC = 3.0 * V * x * x / (E21 * E31 * E41);      /* 12b */
        const double S = 1.0 / E21 + 1.0 / E31 + 1.0 / E41;
        w[0] = C * (4.0 - x * S);                                   /* 12c */
        dw[0] = dC * (4.0 - x * S) - C * S;                         /* 12d (G1) */
        const double Ej1[3] = {E21, E31, E41};
        for (int j = 1; j < 4; j++) {
            w[j] = C * x / Ej1[j - 1];                              /* 12e */
            dw[j] = dC * x / Ej1[j - 1] + C / Ej1[j - 1];           /* 12f (G2) */
        }
        return 1;
    }
    if (E < E3) { /* Eq. 13a-n */
        const double C1 = V * (E - E1) * (E - E1) / (E31 * E41);                    /* 13a */
        const double dC1 = 2.0 * V * (E - E1) / (E31 * E41);                        /* 13b */
        const double C2 = V * (E - E1) * (E - E2) * (E3 - E) / (E31 * E32 * E41);   /* 13c */
        const double dC2 = V / (E31 * E32 * E41) *
                           ((E - E1) * (E2 - E) + (E - E1) * (E3 - E) + (E - E2) * (E3 - E)); /* 13d */
        const double C3 = V * (E - E2) * (E - E2) * (E4 - E) / (E32 * E41 * E42);   /* 13e */
        const double dC3 = V * (E - E2) / (E32 * E41 * E42) * (2.0 * (E4 - E) + (E2 - E)); /* 13f */
        w[0] = C1 + (C1 + C2) * (E3 - E) / E31 + (C1 + C2 + C3) * (E4 - E) / E41;   /* 13g */
        dw[0] = dC1 + (dC1 + dC2) * (E3 - E) / E31 - (C1 + C2) / E31 +
                (dC1 + dC2 + dC3) * (E4 - E) / E41 - (C1 + C2 + C3) / E41;          /* 13h */
        w[1] = C1 + C2 + C3 + (C2 + C3) * (E3 - E) / E32 + C3 * (E4 - E) / E42;     /* 13i */
        dw[1] = dC1 + dC2 + dC3 + (dC2 + dC3) * (E3 - E) / E32 - (C2 + C3) / E32 +
                dC3 * (E4 - E) / E42 - C3 / E42;                                    /* 13j */
        w[2] = (C1 + C2) * (E - E1) / E31 + (C2 + C3) * (E - E2) / E32;             /* 13k (G3) */
        dw[2] = (dC1 + dC2) * (E - E1) / E31 + (C1 + C2) / E31 +
                (dC2 + dC3) * (E - E2) / E32 + (C2 + C3) / E32;                     /* 13l (G4) */
        w[3] = (C1 + C2 + C3) * (E - E1) / E41 + C3 * (E - E2) / E42;               /* 13m */
        dw[3] = (dC1 + dC2 + dC3) * (E - E1) / E41 + (C1 + C2 + C3) / E41 +
                dC3 * (E - E2) / E42 + C3 / E42;                                    /* 13n */
        return 2;
    }
    if (E < E4) { /* Eq. 14a-f */
        const double y = E4 - E;
        const double C = V * y * y * y / (E41 * E42 * E43);         /* 14a */
        const double dC = -3.0 * V * y * y / (E41 * E42 * E43);     /* 14b */
        const double S = 1.0 / E41 + 1.0 / E42 + 1.0 / E43;
        const double E4j[3] = {E41, E42, E43};
        for (int j = 0; j < 3; j++) {
            w[j] = V - C * y / E4j[j];                              /* 14c */
            dw[j] = -dC * y / E4j[j] + C / E4j[j];                  /* 14d */
        }
        w[3] = V - C * (4.0 - S * y);                               /* 14e (G5) */
        dw[3] = -dC * (4.0 - S * y) - C * S;                        /* 14f (G5) */
        return 3;
    }
    for (int j = 0; j < 4; j++) { /* Eq. 15 */
        w[j] = V;
        dw[j] = 0.0;
    }
    return 4;
}

static inline double get_E(const float* E, int layout, long nk, int nb, long ik, int n) {
    return layout == ORACLE_AOS ? (double)E[ik * nb + n] : (double)E[(long)n * nk + ik];
}
static inline double get_W(const float* W, int layout, long nk, int nb, int norb, long ik, int n, int m) {
    if (!W) return 1.0; /* W == NULL: total DOS, X = 1 */
    return layout == ORACLE_AOS ? (double)W[(ik * nb + n) * norb + m]
                                : (double)W[((long)n * norb + m) * nk + ik];
}

/* first index i with omega[i] >= x (nE if none) -- used only by the windowed variant */
static int lower_bound_f(const float* om, int nE, double x) {
    int lo = 0, hi = nE;
    while (lo < hi) {
        int mid = (lo + hi) / 2;
        if ((double)om[mid] < x) lo = mid + 1; else hi = mid;
    }
    return lo;
}
/* first index i with omega[i] > x */
static int upper_bound_f(const float* om, int nE, double x) {
    int lo = 0, hi = nE;
    while (lo < hi) {
        int mid = (lo + hi) / 2;
        if ((double)om[mid] <= x) lo = mid + 1; else hi = mid;
    }
    return lo;
}

/*
 * The whole path.
 *
 *  E, W     fp32 inputs exactly as the CUDA path receives them (widened to double here);
 *           W == NULL means W == 1 with norb == 1.
 *  nk[3]    grid N1, N2, N3 (each >= 1 here; periodic).  ik = ix + N1*(iy + N2*iz).
 *  omega    nE energies (any order is fine for the literal variant).
 *  cube_lo, cube_hi   half-open range of linear cube indices to process (the cube at
 *           k-point ik has its corner 1 there); pass 0, N1*N2*N3 for the full zone.
 *           A sub-range gives that range's additive share of DOS and N.
 *  windowed 0: literal -- every omega for every (tetrahedron, band), Eq. 11/15 included.
 *           1: only omega with E1 < w < E4 are evaluated with Eq. 12-14; the Eq. 15
 *              constant V*b for w >= E4 is added once into a step array at the first such
 *              energy and prefix-summed at the end (needs omega ascending).  Validated
 *              against the literal variant in tests/test_oracle_pins.py.
 *  nthreads 1: strictly sequential, cubes in ik order.  >1: OpenMP over cubes with one
 *              private fp64 histogram per thread, summed at the end (the sum over
 *              tetrahedra of Eq. 9 has no prescribed order).
 *  dos, nos out [norb][nE] doubles, overwritten.
 *  counters out (may be NULL): [0] n_tb = (tetrahedron, band) pairs visited,
 *           [1] n_eval = #(tb, w) with E1 < w < E4, [2..4] evaluations in Eq. 12 / 13 / 14.
 * Returns 0, or -1 on bad arguments / allocation failure.
 */
int oracle_tetra_dos(const float* E, const float* W, const int nk[3], int nb, int norb, int layout,
                     const float* omega, int nE, long cube_lo, long cube_hi, int windowed,
                     int nthreads, double* dos, double* nos, long long* counters) {
    if (!E || !omega || !dos || !nos || !nk) return -1;
    const int N1 = nk[0], N2 = nk[1], N3 = nk[2];
    if (N1 < 1 || N2 < 1 || N3 < 1 || nb < 1 || norb < 1 || nE < 1) return -1;
    if (!W && norb != 1) return -1;
    const long nkt = (long)N1 * N2 * N3;
    if (cube_lo < 0 || cube_hi > nkt || cube_lo > cube_hi) return -1;
    if (nthreads < 1) nthreads = 1;
#ifndef _OPENMP
    nthreads = 1;
#endif
    const double V = 1.0 / (24.0 * (double)nkt); /* V_T/(4 V_G), reading G9 */
    const size_t hist = (size_t)norb * nE;

    /* per-thread histograms: DOS, N and (windowed only) the Eq.-15 step array */
    double* buf = (double*)calloc((size_t)nthreads * 3 * hist, sizeof(double));
    long long* cnt = (long long*)calloc((size_t)nthreads * 8, sizeof(long long));
    if (!buf || !cnt) { free(buf); free(cnt); return -1; }

#ifdef _OPENMP
#pragma omp parallel num_threads(nthreads)
#endif
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        double* D = buf + (size_t)tid * 3 * hist;
        double* Nn = D + hist;
        double* St = Nn + hist;
        long long* c = cnt + (size_t)tid * 8;
        double* b = (double*)malloc(sizeof(double) * 4 * norb); /* b[l][m], sorted corner order */

#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (long cube = cube_lo; cube < cube_hi; cube++) {
            const int ix = (int)(cube % N1), iy = (int)((cube / N1) % N2), iz = (int)(cube / ((long)N1 * N2));
            /* step 2: the 8 corners of the cube, periodic wrap (G7, G8) */
            long corner_ik[9];
            for (int cl = 1; cl <= 8; cl++) {
                int d[3];
                oracle_corner_offset(cl, d);
                const int jx = (ix + d[0]) % N1, jy = (iy + d[1]) % N2, jz = (iz + d[2]) % N3;
                corner_ik[cl] = jx + (long)N1 * (jy + (long)N2 * jz);
            }
            /* step 3: six tetrahedra of Table I, every band */
            for (int t = 0; t < 6; t++) {
                for (int n = 0; n < nb; n++) {
                    double e_in[4], e[4];
                    int perm[4];
                    for (int j = 0; j < 4; j++) e_in[j] = get_E(E, layout, nkt, nb, corner_ik[TABLE_I[t][j]], n);
                    oracle_sort4(e_in, e, perm);
                    for (int l = 0; l < 4; l++)
                        for (int m = 0; m < norb; m++)
                            b[l * norb + m] = get_W(W, layout, nkt, nb, norb, corner_ik[TABLE_I[t][perm[l]]], n, m);
                    c[0]++;
                    int i_lo = 0, i_hi = nE;
                    if (windowed) {
                        i_lo = upper_bound_f(omega, nE, e[0]); /* first w > E1 */
                        /* first w for which Eq. 15 applies: w >= E4, and w > E1 (test order G10) */
                        i_hi = (e[3] > e[0]) ? lower_bound_f(omega, nE, e[3]) : i_lo;
                        if (i_hi < nE)
                            for (int m = 0; m < norb; m++) {
                                double s = 0.0;
                                for (int l = 0; l < 4; l++) s += b[l * norb + m] * V;
                                St[(size_t)m * nE + i_hi] += s;
                            }
                    }
                    /* steps 4-5: every energy of interest */
                    for (int i = i_lo; i < i_hi; i++) {
                        double w[4], dw[4];
                        const double Ei = (double)omega[i];
                        const int kase = oracle_corner_weights(e, Ei, V, w, dw);
                        if (kase >= 1 && kase <= 3) { c[1]++; c[1 + kase]++; }
                        if (kase == 0) continue; /* Eq. 11: nothing to add */
                        for (int m = 0; m < norb; m++) {
                            double T = 0.0, nm = 0.0;
                            for (int l = 0; l < 4; l++) {
                                T += b[l * norb + m] * dw[l];  /* Eq. 8 */
                                nm += b[l * norb + m] * w[l];  /* Eq. 2-3 with Eq. 7 */
                            }
                            D[(size_t)m * nE + i] += T;         /* Eq. 9 */
                            Nn[(size_t)m * nE + i] += nm;
                        }
                    }
                }
            }
        }
        free(b);
    }

    memset(dos, 0, hist * sizeof(double));
    memset(nos, 0, hist * sizeof(double));
    double* step = (double*)calloc(hist, sizeof(double));
    if (!step) { free(buf); free(cnt); return -1; }
    for (int t = 0; t < nthreads; t++) {
        const double* D = buf + (size_t)t * 3 * hist;
        for (size_t j = 0; j < hist; j++) {
            dos[j] += D[j];
            nos[j] += D[hist + j];
            step[j] += D[2 * hist + j];
        }
    }
    if (windowed)
        for (int m = 0; m < norb; m++) {
            double run = 0.0;
            for (int i = 0; i < nE; i++) {
                run += step[(size_t)m * nE + i];
                nos[(size_t)m * nE + i] += run;
            }
        }
    if (counters) {
        for (int j = 0; j < 5; j++) counters[j] = 0;
        for (int t = 0; t < nthreads; t++)
            for (int j = 0; j < 5; j++) counters[j] += cnt[(size_t)t * 8 + j];
    }
    free(step);
    free(buf);
    free(cnt);
    return 0;
}

/* Number of hardware threads OpenMP would use (for the cpu_baseline "cores" field). */
int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * Generic tetrahedron integration weights (Eq. 5-7, :58-71): for every k-point j and band n,
 *     wk[e][n][j] = sum over the tetrahedra T that have j as a corner of w_{n,l(j,T)}(E_e),
 * so that <X>(E_e) = sum_n sum_j X_n(k_j) wk[e][n][j] for any X (Eq. 7), and dwk the same with dw/dE
 * (X = b_{n,m} gives N_m and DOS_m of oracle_tetra_dos: that identity is the pin of this routine's
 * corner <-> k-point bookkeeping, tests/test_oracle_pins.py).  Same cubes, Table I, wrap, sort and
 * test order as oracle_tetra_dos; strictly sequential; the literal Eq. 11-15 for every energy.
 * wk, dwk: out [nW][nb][nk] doubles (k fastest), overwritten; dwk may be NULL.
 */
int oracle_tetra_weights(const float* E, const int nk3[3], int nb, int layout, const float* energies, int nW,
                         double* wk, double* dwk) {
    if (!E || !nk3 || !energies || !wk || nb < 1 || nW < 1) return -1;
    const int N1 = nk3[0], N2 = nk3[1], N3 = nk3[2];
    if (N1 < 1 || N2 < 1 || N3 < 1) return -1;
    const long nk = (long)N1 * N2 * N3;
    const double V = 1.0 / (24.0 * (double)nk); /* G9: V_T/(4 V_G) */
    memset(wk, 0, sizeof(double) * (size_t)nW * nb * nk);
    if (dwk) memset(dwk, 0, sizeof(double) * (size_t)nW * nb * nk);
    for (long cube = 0; cube < nk; cube++) {
        const int ix = (int)(cube % N1), iy = (int)((cube / N1) % N2), iz = (int)(cube / ((long)N1 * N2));
        long corner[8];
        for (int c = 1; c <= 8; c++) {
            int d[3];
            oracle_corner_offset(c, d);
            corner[c - 1] = (long)((ix + d[0]) % N1) + (long)N1 * (((iy + d[1]) % N2) + (long)N2 * ((iz + d[2]) % N3));
        }
        for (int i = 0; i < 6; i++)
            for (int n = 0; n < nb; n++) {
                double e_in[4], e[4], w[4], dw[4];
                int perm[4];
                long kk[4];
                for (int l = 0; l < 4; l++) {
                    kk[l] = corner[TABLE_I[i][l] - 1];
                    e_in[l] = get_E(E, layout, nk, nb, kk[l], n);
                }
                oracle_sort4(e_in, e, perm);
                for (int q = 0; q < nW; q++) {
                    oracle_corner_weights(e, (double)energies[q], V, w, dw);
                    for (int l = 0; l < 4; l++) {
                        const size_t o = ((size_t)q * nb + n) * nk + kk[perm[l]];
                        wk[o] += w[l];
                        if (dwk) dwk[o] += dw[l];
                    }
                }
            }
    }
    return 0;
}
