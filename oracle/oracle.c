/* oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU statement of what the tdx hot path computes, written from
 * /root/reference/PAPER.md (Ha, Park & You, arxiv 1812.01178) and the readings listed in DESIGN.md.
 * fp64 throughout (the paper's precision: cusparseDgtsv), true divisions, no FMA
 * contraction (built with -ffp-contract=off), no blocking/fusion/reordering beyond the cited formulas.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
 * this library.  It shares no code, header, table or constant with paper_1812_01178_b200/csrc.
 *
 * Every function is pinned by tests/test_oracle_pins.py (dense Gaussian elimination, manufactured
 * solutions, eigen closed forms, the printed structure of Z and Z-bar at PAPER.md:L116/L136, the
 * dominance invariants at L162/L172) and tests/test_oracle_partition_pins.py (PDD / PPT step by step; PDD on a
 * periodic line, oracle_cyclic_pdd_line, against a dense LAPACK Woodbury restatement with the far spike ends deleted,
 * the block spike equations, exactness when decayed).  Nothing here is "parity unpinned".
 *
 * Layout of 3-D fields: x fastest, idx(i,j,k) = i + nx*(j + ny*k); all solves in place.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR (-1)

enum { BC_DIRICHLET = 0, BC_PERIODIC = 1, BC_NEUMANN = 2 };
enum { MODE_THOMAS = 0, MODE_PDD = 1, MODE_PPT = 2 };

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Thread count of the OpenMP loops over lines (bench.py's cpu_baseline quotes an all-cores and a 1-thread figure,
 * SURVEY 8(d)); no arithmetic depends on it: every line is solved by one thread, start to end. */
int oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n;
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * Partition map (reading A5; the paper only has m = n/p).
 * q = floor(n/P), r = n mod P, start_p = p*q + min(p,r); partition p owns rows [start_p, start_{p+1}).
 * ------------------------------------------------------------------------------------------- */
int oracle_partition_bounds(int n, int P, int *starts) {
    if (n < 2 || P < 1 || n / P < 2) return ORACLE_ERR;
    int q = n / P, r = n % P;
    for (int p = 0; p <= P; ++p) starts[p] = p * q + (p < r ? p : r);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * Grid metrics (reading A3; PAPER.md:L41 staggered grid, L45 second-order central).
 * faces f_0<...<f_n.  width D_j = f_{j+1}-f_j, centre c_j = (f_j+f_{j+1})/2,
 * hm_j = c_j-c_{j-1}, hp_j = c_{j+1}-c_j; mirrored ghost at the ends: hm_0 = D_0, hp_{n-1} = D_{n-1};
 * periodic: hm_0 = hp_{n-1} = (D_0+D_{n-1})/2.
 * delta2 u_j = [ (u_{j+1}-u_j)/hp_j - (u_j-u_{j-1})/hm_j ] / D_j,  lo_j = 1/(hm_j D_j), up_j = 1/(hp_j D_j).
 * ------------------------------------------------------------------------------------------- */
int oracle_metrics(int n, const double *f, int bc, double *lo, double *up) {
    if (n < 2) return ORACLE_ERR;
    for (int j = 0; j < n; ++j) {
        double D = f[j + 1] - f[j];
        if (!(D > 0.0)) return ORACLE_ERR;
        double hm, hp;
        if (j > 0) hm = 0.5 * (f[j] + f[j + 1]) - 0.5 * (f[j - 1] + f[j]);
        else hm = (bc == BC_PERIODIC) ? 0.5 * ((f[1] - f[0]) + (f[n] - f[n - 1])) : D;
        if (j < n - 1) hp = 0.5 * (f[j + 1] + f[j + 2]) - 0.5 * (f[j] + f[j + 1]);
        else hp = (bc == BC_PERIODIC) ? 0.5 * ((f[1] - f[0]) + (f[n] - f[n - 1])) : D;
        lo[j] = 1.0 / (hm * D);
        up[j] = 1.0 / (hp * D);
    }
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * ADI operator (I - alpha*delta2) (|b_j| = |a_j|+|c_j|+1).
 * a_j = -alpha*lo_j, c_j = -alpha*up_j, b_j = 1 - a_j - c_j on every row.
 * Dirichlet ends: ghost coupling dropped, a_0 := 0, c_{n-1} := 0, b unchanged (reading A3).
 * Neumann ends: ghost mirrors the end cell, so its coupling folds into b: b_0 := 1 - c_0, a_0 := 0,
 *               b_{n-1} := 1 - a_{n-1}, c_{n-1} := 0.
 * Periodic: a_0 couples to row n-1, c_{n-1} to row 0 (kept in a[0], c[n-1]).
 * ------------------------------------------------------------------------------------------- */
int oracle_adi_coeffs(int n, const double *f, int bc, double alpha, double *a, double *b, double *c) {
    double *lo = (double *)malloc(sizeof(double) * n), *up = (double *)malloc(sizeof(double) * n);
    if (oracle_metrics(n, f, bc, lo, up) != ORACLE_OK) { free(lo); free(up); return ORACLE_ERR; }
    for (int j = 0; j < n; ++j) {
        a[j] = -alpha * lo[j];
        c[j] = -alpha * up[j];
        b[j] = 1.0 - a[j] - c[j];
    }
    if (bc == BC_DIRICHLET) { a[0] = 0.0; c[n - 1] = 0.0; }
    if (bc == BC_NEUMANN) { b[0] = 1.0 - c[0]; a[0] = 0.0; b[n - 1] = 1.0 - a[n - 1]; c[n - 1] = 0.0; }
    free(lo); free(up);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * Face-located unknowns ("velocity components at cell faces": the wall-normal
 * component of the ADI step lives on the y-faces).  Row i of a line holds the value at face f_{i+1}, i = 0..n-1.
 * Second difference at a face from the two adjacent CELL widths Db = f_{i+1}-f_i (below), Da = f_{i+2}-f_{i+1}
 * (above) and the distance between the adjacent cell centres hc = (Db+Da)/2:
 *   delta2 v_i = [ (v_{i+1}-v_i)/Da - (v_i-v_{i-1})/Db ] / hc,   lo_i = 1/(Db hc), up_i = 1/(Da hc)
 * (exact for quadratics on any grid).  Dirichlet: the walls f_0 and f_n carry v = 0; row n-1 IS the wall face f_n and
 * is an identity row (lo = up = 0), rows 0 and n-2 lose their wall coupling (b unchanged).  Periodic: face f_n is
 * face f_0, every row is regular, Da of row n-1 wraps to f_1-f_0.  Neumann is not defined for face unknowns.
 * ------------------------------------------------------------------------------------------- */
int oracle_metrics_face(int n, const double *f, int bc, double *lo, double *up) {
    if (n < 3 || bc == BC_NEUMANN) return ORACLE_ERR;
    for (int i = 0; i < n; ++i) {
        if (bc == BC_DIRICHLET && i == n - 1) { lo[i] = 0.0; up[i] = 0.0; continue; }
        double Db = f[i + 1] - f[i];
        double Da = (i + 2 <= n) ? f[i + 2] - f[i + 1] : f[1] - f[0];
        if (!(Db > 0.0) || !(Da > 0.0)) return ORACLE_ERR;
        double hc = 0.5 * (Db + Da);
        lo[i] = 1.0 / (Db * hc);
        up[i] = 1.0 / (Da * hc);
    }
    return ORACLE_OK;
}

/* ADI rows for face unknowns: a = -alpha lo, c = -alpha up, b = 1 - a - c; Dirichlet: a_0 := 0, c_{n-2} := 0 (wall
 * values are 0), row n-1 is the identity. */
int oracle_adi_coeffs_face(int n, const double *f, int bc, double alpha, double *a, double *b, double *c) {
    double *lo = (double *)malloc(sizeof(double) * n), *up = (double *)malloc(sizeof(double) * n);
    if (oracle_metrics_face(n, f, bc, lo, up) != ORACLE_OK) { free(lo); free(up); return ORACLE_ERR; }
    for (int j = 0; j < n; ++j) {
        a[j] = -alpha * lo[j];
        c[j] = -alpha * up[j];
        b[j] = 1.0 - a[j] - c[j];
    }
    if (bc == BC_DIRICHLET) { a[0] = 0.0; c[n - 2] = 0.0; }
    free(lo); free(up);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * Helmholtz operator (delta2_y - lambda), lambda >= 0 (main diagonal = off-diagonal sum
 * plus modified wavenumbers, |b_j| = |a_j|+|c_j|+eps with eps = lambda).
 * a_j = lo_j, c_j = up_j, b_j = -(a_j+c_j) - lambda.  Neumann ends (pseudo-pressure):
 * b_0 = -c_0 - lambda, a_0 := 0; b_{n-1} = -a_{n-1} - lambda, c_{n-1} := 0.
 * lambda == 0 exactly is singular: pin row 0, b_0 := 1, c_0 := 0 (and the caller sets d_0 := 0);
 * *pinned reports it (BASELINE.json config 2: "kz=0 mode pinned at one point").
 * ------------------------------------------------------------------------------------------- */
int oracle_helmholtz_coeffs(int n, const double *f, double lambda, double *a, double *b, double *c, int *pinned) {
    double *lo = (double *)malloc(sizeof(double) * n), *up = (double *)malloc(sizeof(double) * n);
    if (oracle_metrics(n, f, BC_NEUMANN, lo, up) != ORACLE_OK) { free(lo); free(up); return ORACLE_ERR; }
    for (int j = 0; j < n; ++j) {
        a[j] = lo[j];
        c[j] = up[j];
        b[j] = -(a[j] + c[j]) - lambda;
    }
    b[0] = -c[0] - lambda; a[0] = 0.0;
    b[n - 1] = -a[n - 1] - lambda; c[n - 1] = 0.0;
    *pinned = 0;
    if (lambda == 0.0) { b[0] = 1.0; c[0] = 0.0; *pinned = 1; }
    free(lo); free(up);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * Thomas algorithm, textbook form: no pivoting, true divisions.
 * c'_0 = c_0/b_0, d'_0 = d_0/b_0; den = b_j - a_j c'_{j-1}; c'_j = c_j/den; d'_j = (d_j - a_j d'_{j-1})/den;
 * x_{n-1} = d'_{n-1}; x_j = d'_j - c'_j x_{j+1}.   a[0] and c[n-1] are ignored.  x may alias d.
 * ------------------------------------------------------------------------------------------- */
int oracle_thomas(int n, const double *a, const double *b, const double *c, const double *d, double *x) {
    double *cp = (double *)malloc(sizeof(double) * n), *dp = (double *)malloc(sizeof(double) * n);
    cp[0] = c[0] / b[0];
    dp[0] = d[0] / b[0];
    for (int j = 1; j < n; ++j) {
        double den = b[j] - a[j] * cp[j - 1];
        cp[j] = c[j] / den;
        dp[j] = (d[j] - a[j] * dp[j - 1]) / den;
    }
    x[n - 1] = dp[n - 1];
    for (int j = n - 2; j >= 0; --j) x[j] = dp[j] - cp[j] * x[j + 1];
    free(cp); free(dp);
    return ORACLE_OK;
}

/* Same recurrence in long double: the arbiter of SURVEY 8(c) C4 for the 1e-12 Helmholtz gate. */
int oracle_thomas_ld(int n, const double *a, const double *b, const double *c, const double *d, double *x) {
    long double *cp = (long double *)malloc(sizeof(long double) * n), *dp = (long double *)malloc(sizeof(long double) * n);
    cp[0] = (long double)c[0] / b[0];
    dp[0] = (long double)d[0] / b[0];
    for (int j = 1; j < n; ++j) {
        long double den = (long double)b[j] - (long double)a[j] * cp[j - 1];
        cp[j] = (long double)c[j] / den;
        dp[j] = ((long double)d[j] - (long double)a[j] * dp[j - 1]) / den;
    }
    long double xn = dp[n - 1];
    x[n - 1] = (double)xn;
    for (int j = n - 2; j >= 0; --j) { xn = dp[j] - cp[j] * xn; x[j] = (double)xn; }
    free(cp); free(dp);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * Cyclic tridiagonal by Sherman-Morrison (identity: PAPER.md Eq.(3) L97-99 with a rank-1 update;
 * periodic z is named by BASELINE.json north_star, not by the paper).
 * A_cyc has a[0] coupling row 0 to row n-1 and c[n-1] coupling row n-1 to row 0.
 * gamma = -b_0; u = (gamma,0,..,0,c_{n-1})^T, v^T = (1,0,..,0,a_0/gamma); A' = A_cyc - u v^T is plain
 * tridiagonal with b'_0 = b_0 - gamma, b'_{n-1} = b_{n-1} - c_{n-1} a_0/gamma.
 * Solve A'y = d, A'q = u; x = y - q (y_0 + (a_0/gamma) y_{n-1}) / (1 + q_0 + (a_0/gamma) q_{n-1}).
 * ------------------------------------------------------------------------------------------- */
static void cyclic_split(int n, const double *a, const double *b, const double *c,
                         double *a2, double *b2, double *c2, double *u, double *g) {
    double gamma = -b[0];
    memcpy(a2, a, sizeof(double) * n); memcpy(b2, b, sizeof(double) * n); memcpy(c2, c, sizeof(double) * n);
    *g = a[0] / gamma;
    b2[0] = b[0] - gamma;
    b2[n - 1] = b[n - 1] - c[n - 1] * (*g);
    a2[0] = 0.0; c2[n - 1] = 0.0;
    memset(u, 0, sizeof(double) * n);
    u[0] = gamma; u[n - 1] = c[n - 1];
}

int oracle_cyclic_thomas(int n, const double *a, const double *b, const double *c, const double *d, double *x) {
    if (n < 3) return ORACLE_ERR;
    double *w = (double *)malloc(sizeof(double) * n * 6);
    double *a2 = w, *b2 = w + n, *c2 = w + 2 * n, *u = w + 3 * n, *y = w + 4 * n, *q = w + 5 * n, g;
    cyclic_split(n, a, b, c, a2, b2, c2, u, &g);
    oracle_thomas(n, a2, b2, c2, d, y);
    oracle_thomas(n, a2, b2, c2, u, q);
    double s = (y[0] + g * y[n - 1]) / (1.0 + q[0] + g * q[n - 1]);
    for (int j = 0; j < n; ++j) x[j] = y[j] - q[j] * s;
    free(w);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * Dense Gaussian elimination with partial pivoting (row-major A, n x n), the pin for everything else
 * on tiny systems (BASELINE.json north_star: "dense Gaussian elimination on tiny grids").
 * A and d are not modified.
 * ------------------------------------------------------------------------------------------- */
int oracle_dense_solve(int n, const double *A, const double *d, double *x) {
    double *M = (double *)malloc(sizeof(double) * n * (n + 1));
    for (int i = 0; i < n; ++i) { memcpy(M + i * (n + 1), A + i * n, sizeof(double) * n); M[i * (n + 1) + n] = d[i]; }
    for (int k = 0; k < n; ++k) {
        int piv = k; double best = fabs(M[k * (n + 1) + k]);
        for (int i = k + 1; i < n; ++i) if (fabs(M[i * (n + 1) + k]) > best) { best = fabs(M[i * (n + 1) + k]); piv = i; }
        if (best == 0.0) { free(M); return ORACLE_ERR; }
        if (piv != k) for (int j = 0; j <= n; ++j) { double t = M[k * (n + 1) + j]; M[k * (n + 1) + j] = M[piv * (n + 1) + j]; M[piv * (n + 1) + j] = t; }
        for (int i = k + 1; i < n; ++i) {
            double f = M[i * (n + 1) + k] / M[k * (n + 1) + k];
            if (f != 0.0) for (int j = k; j <= n; ++j) M[i * (n + 1) + j] -= f * M[k * (n + 1) + j];
        }
    }
    for (int i = n - 1; i >= 0; --i) {
        double s = M[i * (n + 1) + n];
        for (int j = i + 1; j < n; ++j) s -= M[i * (n + 1) + j] * x[j];
        x[i] = s / M[i * (n + 1) + i];
    }
    free(M);
    return ORACLE_OK;
}

/* Dense matrix of a (cyclic) tridiagonal system, row-major, for manufactured-solution tests: d = A x. */
int oracle_dense_from_tridiag(int n, const double *a, const double *b, const double *c, int cyclic, double *A) {
    memset(A, 0, sizeof(double) * n * n);
    for (int j = 0; j < n; ++j) {
        A[j * n + j] = b[j];
        if (j > 0) A[j * n + j - 1] = a[j];
        if (j < n - 1) A[j * n + j + 1] = c[j];
    }
    if (cyclic) { A[0 * n + n - 1] += a[0]; A[(n - 1) * n + 0] += c[n - 1]; }
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * PDD / PPT, step by step in the paper's order and notation (Eqs.(3)-(11);
 * re-derivation of the garbled matrices: DESIGN.md readings A1, A2).  0-based partitions p=0..P-1,
 * first_p = start_p, last_p = start_{p+1}-1.
 *
 *  A = A~ + dA,  dA = V E^T holds a_{first_i} at (first_i, last_{i-1}) and c_{last_{i-1}} at (last_{i-1}, first_i)
 *  for every interface i = 1..P-1 (L78-91).  A~ is block diagonal with blocks A_p = rows of partition p with
 *  a_first, c_last zeroed (Algorithm 1 step 2, L237-239).
 *  Eq.(5)  A~ x~ = d           -> xt  (per-partition Thomas)
 *  Eq.(6)  A~ Y  = V           -> v^(p) = A_p^{-1}(a_first e_first) (p>=1),  w^(p) = A_p^{-1}(c_last e_last) (p<=P-2)
 *  Z = I + E^T A~^{-1} V  (L112-116), unknowns y_{2i-1} = x_{last_{i-1}}, y_{2i} = x_{first_i} (1-based y):
 *      row 2i-1:  v_last^(i-1) y_{2i-3} + y_{2i-1} + w_last^(i-1) y_{2i}   = xt_{last_{i-1}}
 *      row 2i  :  v_first^(i)  y_{2i-1} + y_{2i}   + w_first^(i)  y_{2i+2} = xt_{first_i}
 *  Eq.(7)  Z y = E^T x~ ;  Eq.(8)  x = x~ - Y y :  x^(p) = xt^(p) - v^(p) y_{2p-1} - w^(p) y_{2p+2}  (0-based p,
 *      y_{-1} = y_{2P} = 0; Algorithm 1 step 7, L257-258).
 *  PPT (L156): Z solved exactly (here: dense GE with partial pivoting; Z-bar = Z P of Eq.(10) is the same
 *      system with columns pair-swapped, see oracle_build_Zbar).
 *  PDD (L148-154): drop v_last^(i-1) in row 2i-1 and w_first^(i) in row 2i; 2x2 blocks solved by the explicit
 *      inverse (Algorithm 1 step 5, L252-254).
 * ------------------------------------------------------------------------------------------- */

/* Eq.(5),(6): local solves. xt, v, w have length n (v zero on partition 0, w zero on partition P-1). */
int oracle_local_solves(int n, int P, const double *a, const double *b, const double *c, const double *d,
                        double *xt, double *v, double *w) {
    int *st = (int *)malloc(sizeof(int) * (P + 1));
    if (oracle_partition_bounds(n, P, st) != ORACLE_OK) { free(st); return ORACLE_ERR; }
    for (int p = 0; p < P; ++p) {
        int s = st[p], m = st[p + 1] - st[p];
        double *aa = (double *)malloc(sizeof(double) * m * 3), *cc = aa + m, *e = aa + 2 * m;
        memcpy(aa, a + s, sizeof(double) * m); memcpy(cc, c + s, sizeof(double) * m);
        aa[0] = 0.0; cc[m - 1] = 0.0;                                   /* Alg.1 step 2 */
        if (d) oracle_thomas(m, aa, b + s, cc, d + s, xt + s);          /* Eq.(5) */
        if (v) {
            memset(e, 0, sizeof(double) * m);
            if (p > 0) { e[0] = a[s]; oracle_thomas(m, aa, b + s, cc, e, v + s); }       /* Eq.(6), a-corner */
            else memset(v + s, 0, sizeof(double) * m);
        }
        if (w) {
            memset(e, 0, sizeof(double) * m);
            if (p < P - 1) { e[m - 1] = c[s + m - 1]; oracle_thomas(m, aa, b + s, cc, e, w + s); } /* c-corner */
            else memset(w + s, 0, sizeof(double) * m);
        }
        free(aa);
    }
    free(st);
    return ORACLE_OK;
}

/* Z of PAPER.md:L116, row-major K x K with K = 2(P-1), from the spikes. pdd != 0 deletes the far-end
 * entries v_last, w_first (L152-154). */
int oracle_build_Z(int n, int P, const double *v, const double *w, int pdd, double *Z) {
    int K = 2 * (P - 1);
    int *st = (int *)malloc(sizeof(int) * (P + 1));
    if (oracle_partition_bounds(n, P, st) != ORACLE_OK) { free(st); return ORACLE_ERR; }
    memset(Z, 0, sizeof(double) * K * K);
    for (int i = 1; i <= P - 1; ++i) {
        int r1 = 2 * i - 2, r2 = 2 * i - 1;                 /* 0-based rows of y_{2i-1}, y_{2i} */
        int last = st[i] - 1, first = st[i];
        Z[r1 * K + r1] = 1.0; Z[r2 * K + r2] = 1.0;
        Z[r1 * K + r2] = w[last];                            /* w_last^(i-1) */
        Z[r2 * K + r1] = v[first];                           /* v_first^(i)  */
        if (!pdd) {
            if (i >= 2) Z[r1 * K + (r1 - 2)] = v[last];      /* v_last^(i-1) * y_{2i-3} */
            if (i <= P - 2) Z[r2 * K + (r2 + 2)] = w[first]; /* w_first^(i)  * y_{2i+2} */
        }
    }
    free(st);
    return ORACLE_OK;
}

/* Z-bar = Z * Pm with Pm the pairwise column swap (1<->2, 3<->4, ...) of PAPER.md:L126-136 (reading A2). */
int oracle_build_Zbar(int K, const double *Z, double *Zbar) {
    for (int r = 0; r < K; ++r)
        for (int cidx = 0; cidx < K; ++cidx) Zbar[r * K + cidx] = Z[r * K + (cidx ^ 1)];
    return ORACLE_OK;
}

/* a-priori PDD bound: dropped = max_i max(|v_last^(i-1)|, |w_first^(i)|) (matrix only). */
double oracle_pdd_dropped(int n, int P, const double *a, const double *b, const double *c) {
    if (P < 2) return 0.0;
    double *v = (double *)malloc(sizeof(double) * n * 2), *w = v + n;
    int *st = (int *)malloc(sizeof(int) * (P + 1));
    double dr = 0.0;
    if (oracle_partition_bounds(n, P, st) == ORACLE_OK && oracle_local_solves(n, P, a, b, c, NULL, NULL, v, w) == ORACLE_OK) {
        for (int i = 1; i <= P - 1; ++i) {
            if (i >= 2 && fabs(v[st[i] - 1]) > dr) dr = fabs(v[st[i] - 1]);
            if (i <= P - 2 && fabs(w[st[i]]) > dr) dr = fabs(w[st[i]]);
        }
    } else dr = -1.0;
    free(v); free(st);
    return dr;
}

/* One line by PDD (mode 1) or PPT (mode 2); mode 0 / P == 1 is plain Thomas. x may alias d.
 * yout (optional, length 2(P-1)) receives the reduced solution for the interface-value pin. */
int oracle_partitioned_line(int n, int P, int mode, const double *a, const double *b, const double *c,
                            const double *d, double *x, double *yout) {
    if (mode == MODE_THOMAS || P == 1) return oracle_thomas(n, a, b, c, d, x);
    int K = 2 * (P - 1);
    int *st = (int *)malloc(sizeof(int) * (P + 1));
    if (oracle_partition_bounds(n, P, st) != ORACLE_OK) { free(st); return ORACLE_ERR; }
    double *xt = (double *)malloc(sizeof(double) * (3 * n + 2 * K)), *v = xt + n, *w = xt + 2 * n, *r = xt + 3 * n, *y = r + K;
    oracle_local_solves(n, P, a, b, c, d, xt, v, w);
    for (int i = 1; i <= P - 1; ++i) { r[2 * i - 2] = xt[st[i] - 1]; r[2 * i - 1] = xt[st[i]]; }   /* E^T x~ */
    if (mode == MODE_PDD) {
        for (int i = 1; i <= P - 1; ++i) {                          /* Alg.1 step 5: explicit 2x2 inverse */
            double wl = w[st[i] - 1], vf = v[st[i]];
            double det = 1.0 - wl * vf;
            y[2 * i - 2] = (r[2 * i - 2] - wl * r[2 * i - 1]) / det;
            y[2 * i - 1] = (r[2 * i - 1] - vf * r[2 * i - 2]) / det;
        }
    } else {
        double *Z = (double *)malloc(sizeof(double) * K * K);
        oracle_build_Z(n, P, v, w, 0, Z);
        int rc = oracle_dense_solve(K, Z, r, y);                    /* Eq.(7) exactly */
        free(Z);
        if (rc != ORACLE_OK) { free(xt); free(st); return ORACLE_ERR; }
    }
    for (int p = 0; p < P; ++p) {                                   /* Eq.(8) / Alg.1 step 7 */
        double yl = (p > 0) ? y[2 * p - 2] : 0.0;                   /* y_{2p-1} (1-based) */
        double yr = (p < P - 1) ? y[2 * p + 1] : 0.0;               /* y_{2p+2} (1-based) */
        for (int j = st[p]; j < st[p + 1]; ++j) x[j] = xt[j] - v[j] * yl - w[j] * yr;
    }
    if (yout) memcpy(yout, y, sizeof(double) * K);
    free(xt); free(st);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * PDD on a periodic line (reading A16; SURVEY 8(c) C2 "close the reduced system cyclically, P
 * interfaces").  The split A = A~ + dA of PAPER.md:L78-91 now also moves the two wrap-around corners into dA:
 * a_0 at (0, n-1) and c_{n-1} at (n-1, 0), so there are P interfaces, interface i (0 <= i < P) lying between
 * partitions (i-1) mod P and i, and every partition p has both spikes (Eq.(6)):
 *     v^(p) = A_p^{-1}(a_first e_first),   w^(p) = A_p^{-1}(c_last e_last).
 * The exact interface rows read (indices of partitions mod P; s_i = x_{last_{i-1}}, t_i = x_{first_i}):
 *     v_last^(i-1) s_{i-1} + s_i + w_last^(i-1) t_i     = xt_{last_{i-1}}
 *     v_first^(i)  s_i     + t_i + w_first^(i)  t_{i+1} = xt_{first_i}
 * PDD (L148-154) deletes the far spike ends v_last, w_first, which leaves P blocks [[1, w_last^(i-1)],[v_first^(i), 1]]
 * solved by the explicit inverse (Algorithm 1 step 5, L252-254); Eq.(8): x^(p) = xt^(p) - v^(p) s_p - w^(p) t_{p+1}.
 * spikes (optional, 2n doubles) returns v then w.
 * ------------------------------------------------------------------------------------------- */
int oracle_cyclic_pdd_line(int n, int P, const double *a, const double *b, const double *c,
                           const double *d, double *x, double *spikes) {
    if (P < 2 || n < 3) return ORACLE_ERR;
    int *st = (int *)malloc(sizeof(int) * (P + 1));
    if (oracle_partition_bounds(n, P, st) != ORACLE_OK) { free(st); return ORACLE_ERR; }
    double *xt = (double *)malloc(sizeof(double) * (3 * n + 2 * P)), *v = xt + n, *w = xt + 2 * n, *sv = xt + 3 * n, *tv = sv + P;
    for (int p = 0; p < P; ++p) {
        int s = st[p], m = st[p + 1] - st[p];
        double *aa = (double *)malloc(sizeof(double) * m * 3), *cc = aa + m, *e = aa + 2 * m;
        memcpy(aa, a + s, sizeof(double) * m); memcpy(cc, c + s, sizeof(double) * m);
        aa[0] = 0.0; cc[m - 1] = 0.0;                                   /* A_p: Alg.1 step 2, wrap corners included */
        oracle_thomas(m, aa, b + s, cc, d + s, xt + s);                 /* Eq.(5) */
        memset(e, 0, sizeof(double) * m); e[0] = a[s];
        oracle_thomas(m, aa, b + s, cc, e, v + s);                      /* Eq.(6), a-corner (a[0] couples to row n-1) */
        memset(e, 0, sizeof(double) * m); e[m - 1] = c[s + m - 1];
        oracle_thomas(m, aa, b + s, cc, e, w + s);                      /* Eq.(6), c-corner (c[n-1] couples to row 0) */
        free(aa);
    }
    for (int i = 0; i < P; ++i) {                                       /* Alg.1 step 5 on each of the P interfaces */
        int pm = (i + P - 1) % P;
        int last = st[pm + 1] - 1, first = st[i];
        double wl = w[last], vf = v[first];
        double det = 1.0 - wl * vf;
        sv[i] = (xt[last] - wl * xt[first]) / det;
        tv[i] = (xt[first] - vf * xt[last]) / det;
    }
    if (spikes) { memcpy(spikes, v, sizeof(double) * n); memcpy(spikes + n, w, sizeof(double) * n); }
    for (int p = 0; p < P; ++p) {                                       /* Eq.(8) / Alg.1 step 7 */
        double yl = sv[p], yr = tv[(p + 1) % P];
        for (int j = st[p]; j < st[p + 1]; ++j) x[j] = xt[j] - v[j] * yl - w[j] * yr;
    }
    free(xt); free(st);
    return ORACLE_OK;
}

/* a-priori bound of the cyclically closed PDD: max over ALL partitions of |v_last^(p)|, |w_first^(p)|. */
double oracle_cyclic_pdd_dropped(int n, int P, const double *a, const double *b, const double *c) {
    if (P < 2) return 0.0;
    double *wk = (double *)malloc(sizeof(double) * n * 4), *d0 = wk, *x0 = wk + n, *sp = wk + 2 * n;
    int *st = (int *)malloc(sizeof(int) * (P + 1));
    double dr = -1.0;
    memset(d0, 0, sizeof(double) * n);
    if (oracle_partition_bounds(n, P, st) == ORACLE_OK && oracle_cyclic_pdd_line(n, P, a, b, c, d0, x0, sp) == ORACLE_OK) {
        dr = 0.0;
        for (int p = 0; p < P; ++p) {
            double vl = fabs(sp[st[p + 1] - 1]), wf = fabs(sp[n + st[p]]);
            if (vl > dr) dr = vl;
            if (wf > dr) dr = wf;
        }
    }
    free(wk); free(st);
    return dr;
}

/* ---------------------------------------------------------------------------------------------
 * The OTHER definition of PDD on a periodic line ("outer Sherman-Morrison (y and q each by the
 * partitioned solve; q is matrix-only)" -- the definition the survey assigns to the oracle; reading A16
 * says why the product takes the cyclically closed one above).  Rank-1 split of Eq.(3) first (cyclic_split:
 * A' = A_cyc - u v^T, plain tridiagonal), then
 *     y = PDD(A') d   step by step (oracle_partitioned_line, P-1 interfaces, Alg.1 steps 3, 5, 7),
 *     q = A'^{-1} u   exactly (matrix-only, plan time),
 *     x = y - q (y_0 + g y_{n-1}) / (1 + q_0 + g q_{n-1}).
 * Unlike the cyclic closure this is exact at P = 1 and has P-1 interfaces; the two differ by O(dropped) (pinned in
 * tests/test_oracle_partition_pins.py on the six config z-operators and on random weakly dominant lines).
 * ------------------------------------------------------------------------------------------- */
int oracle_cyclic_pdd_outer_line(int n, int P, const double *a, const double *b, const double *c,
                                 const double *d, double *x) {
    if (n < 3) return ORACLE_ERR;
    double *wk = (double *)malloc(sizeof(double) * n * 7);
    double *a2 = wk, *b2 = wk + n, *c2 = wk + 2 * n, *u = wk + 3 * n, *y = wk + 4 * n, *q = wk + 5 * n, *dd = wk + 6 * n, g;
    memcpy(dd, d, sizeof(double) * n);                                   /* x may alias d */
    cyclic_split(n, a, b, c, a2, b2, c2, u, &g);
    int rc = oracle_partitioned_line(n, P, MODE_PDD, a2, b2, c2, dd, y, NULL);
    oracle_thomas(n, a2, b2, c2, u, q);
    double s = (y[0] + g * y[n - 1]) / (1.0 + q[0] + g * q[n - 1]);
    for (int j = 0; j < n; ++j) x[j] = y[j] - q[j] * s;
    free(wk);
    return rc;
}

/* a-priori bound of the outer-split PDD: the far spike ends of A' = the non-periodic bound on the split matrix. */
double oracle_cyclic_pdd_outer_dropped(int n, int P, const double *a, const double *b, const double *c) {
    if (n < 3) return -1.0;
    double *wk = (double *)malloc(sizeof(double) * n * 4), g;
    cyclic_split(n, a, b, c, wk, wk + n, wk + 2 * n, wk + 3 * n, &g);
    double dr = oracle_pdd_dropped(n, P, wk, wk + n, wk + 2 * n);
    free(wk);
    return dr;
}

/* Cyclic line with partitions.  PDD: the cyclically closed reduced system above.  PPT (exact in either form):
 * outer Sherman-Morrison; y = A'^{-1} d by the partitioned solve, q = A'^{-1} u by Thomas. */
int oracle_cyclic_line(int n, int P, int mode, const double *a, const double *b, const double *c,
                       const double *d, double *x) {
    if (mode == MODE_THOMAS || P == 1) return oracle_cyclic_thomas(n, a, b, c, d, x);
    if (mode == MODE_PDD) {
        double *dd = (double *)malloc(sizeof(double) * n);
        memcpy(dd, d, sizeof(double) * n);                               /* x may alias d */
        int rc = oracle_cyclic_pdd_line(n, P, a, b, c, dd, x, NULL);
        free(dd);
        return rc;
    }
    double *wk = (double *)malloc(sizeof(double) * n * 6);
    double *a2 = wk, *b2 = wk + n, *c2 = wk + 2 * n, *u = wk + 3 * n, *y = wk + 4 * n, *q = wk + 5 * n, g;
    cyclic_split(n, a, b, c, a2, b2, c2, u, &g);
    int rc = oracle_partitioned_line(n, P, mode, a2, b2, c2, d, y, NULL);
    oracle_thomas(n, a2, b2, c2, u, q);
    double s = (y[0] + g * y[n - 1]) / (1.0 + q[0] + g * q[n - 1]);
    for (int j = 0; j < n; ++j) x[j] = y[j] - q[j] * s;
    free(wk);
    return rc;
}

/* ---------------------------------------------------------------------------------------------
 * 3-D sweeps: gather one line -> solve -> scatter; OpenMP over lines only.
 * mode: 0 Thomas (cyclic Thomas when periodic), 1 PDD, 2 PPT, 3 Thomas in long double (arbiter; non-periodic).
 * ------------------------------------------------------------------------------------------- */
enum { MODE_THOMAS_LD = 3 };

static int solve_line(int n, int P, int mode, int periodic, const double *a, const double *b, const double *c,
                      double *buf) {
    if (mode == MODE_THOMAS_LD) return periodic ? ORACLE_ERR : oracle_thomas_ld(n, a, b, c, buf, buf);
    if (periodic) return oracle_cyclic_line(n, P, mode, a, b, c, buf, buf);
    return oracle_partitioned_line(n, P, mode, a, b, c, buf, buf, NULL);
}

/* All lines of direction dir (0 x, 1 y, 2 z) share the matrix (a,b,c) of length n_dir. */
int oracle_sweep_coeffs(int nx, int ny, int nz, int dir, int mode, int P, int periodic,
                        const double *a, const double *b, const double *c, double *field) {
    int n = dir == 0 ? nx : (dir == 1 ? ny : nz);
    long stride = dir == 0 ? 1 : (dir == 1 ? (long)nx : (long)nx * ny);
    long nlines = (long)nx * ny * nz / n;
    int err = 0;
    if (mode != MODE_THOMAS && mode != MODE_THOMAS_LD) { int *st = (int *)malloc(sizeof(int) * (P + 1)); int rc = oracle_partition_bounds(n, P, st); free(st); if (rc) return ORACLE_ERR; }
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * n);
#pragma omp for schedule(static)
        for (long l = 0; l < nlines; ++l) {
            long base;
            if (dir == 0) base = l * nx;
            else if (dir == 1) base = (l / nx) * (long)nx * ny + (l % nx);
            else base = l;
            for (int j = 0; j < n; ++j) buf[j] = field[base + j * stride];
            if (solve_line(n, P, mode, periodic, a, b, c, buf) != ORACLE_OK) {
#pragma omp atomic write
                err = 1;
            }
            for (int j = 0; j < n; ++j) field[base + j * stride] = buf[j];
        }
        free(buf);
    }
    return err ? ORACLE_ERR : ORACLE_OK;
}

/* (I - alpha*delta2_dir) x = rhs for every line of direction dir, in place (tdx_adi_sweep's definition). */
int oracle_adi_sweep(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf,
                     int bcx, int bcy, int bcz, int dir, int mode, int P, double alpha, double *field) {
    int n = dir == 0 ? nx : (dir == 1 ? ny : nz);
    const double *f = dir == 0 ? xf : (dir == 1 ? yf : zf);
    int bc = dir == 0 ? bcx : (dir == 1 ? bcy : bcz);
    double *a = (double *)malloc(sizeof(double) * n * 3), *b = a + n, *c = a + 2 * n;
    int rc = oracle_adi_coeffs(n, f, bc, alpha, a, b, c);
    if (rc == ORACLE_OK) rc = oracle_sweep_coeffs(nx, ny, nz, dir, mode, P, bc == BC_PERIODIC, a, b, c, field);
    free(a);
    return rc;
}

/* The same with the unknowns of direction dir at cell centres (loc = 0) or at faces (loc = 1): tdx_adi_sweep_at. */
int oracle_adi_sweep_at(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf,
                        int bcx, int bcy, int bcz, int dir, int loc, int mode, int P, double alpha, double *field) {
    if (loc == 0) return oracle_adi_sweep(nx, ny, nz, xf, yf, zf, bcx, bcy, bcz, dir, mode, P, alpha, field);
    int n = dir == 0 ? nx : (dir == 1 ? ny : nz);
    const double *f = dir == 0 ? xf : (dir == 1 ? yf : zf);
    int bc = dir == 0 ? bcx : (dir == 1 ? bcy : bcz);
    double *a = (double *)malloc(sizeof(double) * n * 3), *b = a + n, *c = a + 2 * n;
    int rc = oracle_adi_coeffs_face(n, f, bc, alpha, a, b, c);
    if (rc == ORACLE_OK) rc = oracle_sweep_coeffs(nx, ny, nz, dir, mode, P, bc == BC_PERIODIC, a, b, c, field);
    free(a);
    return rc;
}

/* General batched cyclic tridiagonal along dir with user coefficients (tdx_cyclic_solve's definition). */
int oracle_cyclic_solve(int nx, int ny, int nz, int dir, int mode, int P,
                        const double *a, const double *b, const double *c, double *field) {
    return oracle_sweep_coeffs(nx, ny, nz, dir, mode, P, 1, a, b, c, field);
}

/* (delta2_y - lambda[i,m]) phi = rhs, lambda = kx2[i] + kz2[m] (kx2 may be NULL = zeros); field is complex128
 * interleaved [nm][ny][nx] (x fastest).  Real matrix, complex RHS: re and im are two real solves with the same
 * matrix ("complex-numbered tridiagonal matrices").  lambda == 0 lines are pinned: d_0 := 0. */
int oracle_helmholtz_solve(int nx, int ny, int nm, const double *yf, const double *kx2, const double *kz2,
                           int mode, int P, double *field) {
    int err = 0;
    if (mode != MODE_THOMAS && mode != MODE_THOMAS_LD) { int *st = (int *)malloc(sizeof(int) * (P + 1)); int rc = oracle_partition_bounds(ny, P, st); free(st); if (rc) return ORACLE_ERR; }
#pragma omp parallel
    {
        double *a = (double *)malloc(sizeof(double) * ny * 5), *b = a + ny, *c = a + 2 * ny, *re = a + 3 * ny, *im = a + 4 * ny;
#pragma omp for schedule(static) collapse(2)
        for (int m = 0; m < nm; ++m)
            for (int i = 0; i < nx; ++i) {
                double lambda = (kx2 ? kx2[i] : 0.0) + kz2[m];
                int pinned;
                if (oracle_helmholtz_coeffs(ny, yf, lambda, a, b, c, &pinned) != ORACLE_OK) {
#pragma omp atomic write
                    err = 1;
                    continue;
                }
                long base = ((long)m * ny * nx + i) * 2;
                for (int j = 0; j < ny; ++j) { re[j] = field[base + (long)j * nx * 2]; im[j] = field[base + (long)j * nx * 2 + 1]; }
                if (pinned) { re[0] = 0.0; im[0] = 0.0; }
                if (solve_line(ny, P, mode, 0, a, b, c, re) != ORACLE_OK || solve_line(ny, P, mode, 0, a, b, c, im) != ORACLE_OK) {
#pragma omp atomic write
                    err = 1;
                }
                for (int j = 0; j < ny; ++j) { field[base + (long)j * nx * 2] = re[j]; field[base + (long)j * nx * 2 + 1] = im[j]; }
            }
        free(a);
    }
    return err ? ORACLE_ERR : ORACLE_OK;
}
