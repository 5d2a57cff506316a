/*
 * cheb_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct FP64 implementation of what the hot path of
 * arXiv 2306.12616 ("A fast, dense Chebyshev solver for electronic structure on GPUs")
 * computes, written from /root/reference/PAPER.md (cited as PAPER.md:<line>).  It shares NO
 * code with the CUDA path (paper_2306_12616_b200/csrc) and must never be imported, linked or
 * executed by the product; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may use it.
 *
 * Style: plain loops in the paper's order and notation.  OpenMP "parallel for" is used only
 * over independent output rows / independent coefficients; it never changes the order in which
 * any single floating-point sum is accumulated.  No blocking, fusion or algebraic reordering.
 *
 * Notation (SURVEY.md notation table; the paper's `m` is called `p` here because
 * BASELINE.json uses m for the number of terms):
 *   N  matrix size                M  number of Chebyshev terms (sum n = 0..M-1; paper's L+1)
 *   k  baby-step block size       p  number of Horner blocks (paper's m), k*p >= M
 *   a,b spectral bounds (eps_a, eps_b)         X = (2H - (a+b)I)/(b-a)
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): see DESIGN.md section "Oracle pins".
 * Every function below is pinned; none is "parity unpinned".
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define CO_PI_L 3.14159265358979323846264338327950288L

int co_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------
 * Eq. (2), PAPER.md:73 -- Fermi-Dirac function f(eps) = 1/(1+exp(beta(eps-mu))),
 * evaluated without overflow: for y = beta(eps-mu) > 0 use e^{-y}/(1+e^{-y}).
 * ---------------------------------------------------------------------------------------- */
double co_fermi(double beta, double mu, double eps) {
    double y = beta * (eps - mu);
    if (y > 0.0) {
        double e = exp(-y);
        return e / (1.0 + e);
    }
    return 1.0 / (1.0 + exp(y));
}

static long double fermi_scaled_l(long double beta_t, long double mu_t, long double x) {
    long double y = beta_t * (x - mu_t);
    if (y > 0.0L) {
        long double e = expl(-y);
        return e / (1.0L + e);
    }
    return 1.0L / (1.0L + expl(y));
}

/* ------------------------------------------------------------------------------------------
 * Plain dense product C = A*B (n x n, row-major), triple loop.  Each C[i][j] is the sum over
 * kk = 0..n-1 in increasing kk (loop order i,kk,j only changes which element is visited when).
 * ---------------------------------------------------------------------------------------- */
void co_matmul(int n, const double* A, const double* B, double* C) {
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n; ++i) {
        double* ci = C + (size_t)i * n;
        for (int j = 0; j < n; ++j) ci[j] = 0.0;
        for (int kk = 0; kk < n; ++kk) {
            double aik = A[(size_t)i * n + kk];
            const double* bk = B + (size_t)kk * n;
            for (int j = 0; j < n; ++j) ci[j] += aik * bk[j];
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * Gershgorin bounds (north_star item 1; the paper assumes eps_a, eps_b known):
 * R_i = sum_{j != i} |h_ij|,  a = min_i (h_ii - R_i),  b = max_i (h_ii + R_i).
 * ---------------------------------------------------------------------------------------- */
void co_gershgorin(int n, const double* H, double* a_out, double* b_out) {
    double a = INFINITY, b = -INFINITY;
    for (int i = 0; i < n; ++i) {
        double R = 0.0;
        for (int j = 0; j < n; ++j)
            if (j != i) R += fabs(H[(size_t)i * n + j]);
        double hii = H[(size_t)i * n + i];
        if (hii - R < a) a = hii - R;
        if (hii + R > b) b = hii + R;
    }
    *a_out = a;
    *b_out = b;
}

/* Scaling of PAPER.md:96 as read in DESIGN.md (reading A1): X = (2H - (a+b) I)/(b-a). */
void co_scale(int n, const double* H, double a, double b, double* X) {
    double inv = 1.0 / (b - a);
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) {
            double h = 2.0 * H[(size_t)i * n + j];
            if (i == j) h -= (a + b);
            X[(size_t)i * n + j] = h * inv;
        }
}

/* ------------------------------------------------------------------------------------------
 * O-eig, step 1: cyclic Jacobi eigendecomposition H = V E V^T of a symmetric matrix
 * (Eq. 1, PAPER.md:65-69 needs the eigenpairs).  Rows of Vt are the eigenvectors.
 * Sweeps over all (p,q), p<q; each rotation annihilates a_pq exactly; stops when
 * off(A) <= tol * ||A||_F.  Returns the number of sweeps, or -1 if not converged.
 * ---------------------------------------------------------------------------------------- */
int co_jacobi_eig(int n, const double* H, double* E, double* Vt, int max_sweeps, double tol) {
    double* A = (double*)malloc(sizeof(double) * (size_t)n * n);
    if (!A) return -2;
    memcpy(A, H, sizeof(double) * (size_t)n * n);
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) Vt[(size_t)i * n + j] = (i == j) ? 1.0 : 0.0;
    double fro2 = 0.0;
    for (size_t t = 0; t < (size_t)n * n; ++t) fro2 += A[t] * A[t];
    int sweep;
    for (sweep = 0; sweep < max_sweeps; ++sweep) {
        double off2 = 0.0;
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < n; ++j)
                if (i != j) off2 += A[(size_t)i * n + j] * A[(size_t)i * n + j];
        if (sqrt(off2) <= tol * sqrt(fro2)) break;
        for (int pp = 0; pp < n - 1; ++pp) {
            for (int q = pp + 1; q < n; ++q) {
                double apq = A[(size_t)pp * n + q];
                if (apq == 0.0) continue;
                double app = A[(size_t)pp * n + pp], aqq = A[(size_t)q * n + q];
                double theta = (aqq - app) / (2.0 * apq);
                double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
                double* rp = A + (size_t)pp * n;
                double* rq = A + (size_t)q * n;
                /* rows p and q of J^T A */
                for (int r = 0; r < n; ++r) {
                    double xp = rp[r], xq = rq[r];
                    rp[r] = c * xp - s * xq;
                    rq[r] = s * xp + c * xq;
                }
                /* columns p and q of (J^T A) J */
                for (int r = 0; r < n; ++r) {
                    double xp = A[(size_t)r * n + pp], xq = A[(size_t)r * n + q];
                    A[(size_t)r * n + pp] = c * xp - s * xq;
                    A[(size_t)r * n + q] = s * xp + c * xq;
                }
                A[(size_t)pp * n + q] = 0.0;
                A[(size_t)q * n + pp] = 0.0;
                double* vp = Vt + (size_t)pp * n;
                double* vq = Vt + (size_t)q * n;
                for (int r = 0; r < n; ++r) {
                    double xp = vp[r], xq = vq[r];
                    vp[r] = c * xp - s * xq;
                    vq[r] = s * xp + c * xq;
                }
            }
        }
    }
    for (int i = 0; i < n; ++i) E[i] = A[(size_t)i * n + i];
    free(A);
    return sweep < max_sweeps ? sweep : -1;
}

/* O-eig, step 2 -- Eq. (1):  D = V f(E) V^T = sum_i f(eps_i) v_i v_i^T. */
void co_dm_from_eig(int n, const double* E, const double* Vt, double beta, double mu, double* D) {
    double* f = (double*)malloc(sizeof(double) * (size_t)n);
    for (int i = 0; i < n; ++i) f[i] = co_fermi(beta, mu, E[i]);
#pragma omp parallel for schedule(static)
    for (int r = 0; r < n; ++r) {
        double* dr = D + (size_t)r * n;
        for (int c = 0; c < n; ++c) dr[c] = 0.0;
        for (int i = 0; i < n; ++i) {
            double w = f[i] * Vt[(size_t)i * n + r];
            const double* vi = Vt + (size_t)i * n;
            for (int c = 0; c < n; ++c) dr[c] += w * vi[c];
        }
    }
    free(f);
}

/* ------------------------------------------------------------------------------------------
 * Chebyshev coefficients of the scaled Fermi function (PAPER.md:91 expansion sum c_n T_n with
 * c_0 NOT halved; the paper is silent on how c_n are obtained -- DESIGN.md reading A3):
 *   beta~ = beta (b-a)/2,  mu~ = (2 mu - (a+b))/(b-a),  f~(x) = 1/(1+exp(beta~ (x - mu~)))
 *   theta_j = pi (j+1/2)/Nq,  x_j = cos theta_j,
 *   c_n = ((2 - delta_n0)/Nq) sum_{j<Nq} f~(x_j) cos(n theta_j),   n < M,
 * with the angle reduced exactly: n theta_j = pi * ((n(2j+1)) mod 4Nq) / (2Nq).
 * Direct O(M Nq) sum in long double.
 * ---------------------------------------------------------------------------------------- */
void co_cheb_coeffs(double beta, double mu, double a, double b, int M, int Nq, double* c) {
    long double beta_t = (long double)beta * ((long double)b - (long double)a) / 2.0L;
    long double mu_t = (2.0L * (long double)mu - ((long double)a + (long double)b)) /
                       ((long double)b - (long double)a);
    long double* fx = (long double*)malloc(sizeof(long double) * (size_t)Nq);
    for (int j = 0; j < Nq; ++j) {
        long double xj = cosl(CO_PI_L * ((long double)j + 0.5L) / (long double)Nq);
        fx[j] = fermi_scaled_l(beta_t, mu_t, xj);
    }
#pragma omp parallel for schedule(static)
    for (int n = 0; n < M; ++n) {
        long double s = 0.0L;
        for (int j = 0; j < Nq; ++j) {
            int64_t r = ((int64_t)n * (2 * (int64_t)j + 1)) % (4 * (int64_t)Nq);
            s += fx[j] * cosl(CO_PI_L * (long double)r / (2.0L * (long double)Nq));
        }
        c[n] = (double)(((n == 0) ? 1.0L : 2.0L) * s / (long double)Nq);
    }
    free(fx);
}

/* Same DCT applied to an arbitrary tabulated function (used only to PIN the DCT itself against
 * closed forms: x^2 -> [1/2, 0, 1/2], T_5 -> e_5).  fvals[j] = f(cos(pi (j+1/2)/Nq)). */
void co_cheb_coeffs_of_samples(const double* fvals, int M, int Nq, double* c) {
    for (int n = 0; n < M; ++n) {
        long double s = 0.0L;
        for (int j = 0; j < Nq; ++j) {
            int64_t r = ((int64_t)n * (2 * (int64_t)j + 1)) % (4 * (int64_t)Nq);
            s += (long double)fvals[j] * cosl(CO_PI_L * (long double)r / (2.0L * (long double)Nq));
        }
        c[n] = (double)(((n == 0) ? 1.0L : 2.0L) * s / (long double)Nq);
    }
}

/* ------------------------------------------------------------------------------------------
 * O-cheb: D_cheb = sum_{n=0}^{M-1} c_n T_n(X) with the three-term recurrence
 * T_0 = I, T_1 = X, T_{n+1} = 2 X T_n - T_{n-1} (the a=1 case of Eq. 7; Eq. 22
 * is its first instance).  M-2 plain products.  If tau != NULL, tau[n] = tr T_n(X), n < M.
 * ---------------------------------------------------------------------------------------- */
void co_dm_cheb(int n, const double* H, double a, double b, const double* c, int M, double* D,
                double* tau) {
    size_t nn = (size_t)n * n;
    double* X = (double*)malloc(sizeof(double) * nn);
    double* Tm = (double*)malloc(sizeof(double) * nn); /* T_{n-1} */
    double* Tc = (double*)malloc(sizeof(double) * nn); /* T_n     */
    double* Tn = (double*)malloc(sizeof(double) * nn); /* T_{n+1} */
    co_scale(n, H, a, b, X);
    for (size_t t = 0; t < nn; ++t) { D[t] = 0.0; Tm[t] = 0.0; }
    for (int i = 0; i < n; ++i) Tm[(size_t)i * n + i] = 1.0;      /* T_0 = I */
    memcpy(Tc, X, sizeof(double) * nn);                            /* T_1 = X */
    for (int t = 0; t < M; ++t) {
        const double* T = (t == 0) ? Tm : Tc;
        if (t >= 2) {
            co_matmul(n, X, Tc, Tn);
            for (size_t e = 0; e < nn; ++e) Tn[e] = 2.0 * Tn[e] - Tm[e];
            double* sw = Tm; Tm = Tc; Tc = Tn; Tn = sw;
            T = Tc;
        }
        for (size_t e = 0; e < nn; ++e) D[e] += c[t] * T[e];
        if (tau) {
            double s = 0.0;
            for (int i = 0; i < n; ++i) s += T[(size_t)i * n + i];
            tau[t] = s;
        }
    }
    free(X); free(Tm); free(Tc); free(Tn);
}

/* Selected columns of D_cheb by the same recurrence applied to unit vectors:
 * v_0 = e_j, v_1 = X e_j, v_{n+1} = 2 X v_n - v_{n-1};  out[s][:] = sum_n c_n v_n.
 * (Column j of sum c_n T_n(X); lets the full-size configs be checked one column at a time.) */
void co_dm_cheb_columns(int n, const double* H, double a, double b, const double* c, int M,
                        int ncols, const int* cols, double* out) {
    size_t nn = (size_t)n * n;
    double* X = (double*)malloc(sizeof(double) * nn);
    co_scale(n, H, a, b, X);
    double* vm = (double*)malloc(sizeof(double) * n);
    double* vc = (double*)malloc(sizeof(double) * n);
    double* vn = (double*)malloc(sizeof(double) * n);
    for (int s = 0; s < ncols; ++s) {
        int j = cols[s];
        double* o = out + (size_t)s * n;
        for (int i = 0; i < n; ++i) { vm[i] = (i == j) ? 1.0 : 0.0; vc[i] = X[(size_t)i * n + j]; o[i] = 0.0; }
        for (int t = 0; t < M; ++t) {
            const double* v = (t == 0) ? vm : vc;
            if (t >= 2) {
#pragma omp parallel for schedule(static)
                for (int i = 0; i < n; ++i) {
                    double acc = 0.0;
                    const double* xi = X + (size_t)i * n;
                    for (int kk = 0; kk < n; ++kk) acc += xi[kk] * vc[kk];
                    vn[i] = 2.0 * acc - vm[i];
                }
                double* sw = vm; vm = vc; vc = vn; vn = sw;
                v = vc;
            }
            for (int i = 0; i < n; ++i) o[i] += c[t] * v[i];
        }
    }
    free(X); free(vm); free(vc); free(vn);
}

/* The same M-term sum applied to arbitrary vectors: out[s] = (sum_{n<M} c_n T_n(X)) V[s], s < nvec, by the
 * three-term recurrence of PAPER.md:91 started from v (w_0 = v, w_1 = X v, w_{n+1} = 2 X w_n - w_{n-1}); no matrix
 * product is formed.  V and out are nvec x n row-major (one vector per row).  With V[s] = e_j this is
 * co_dm_cheb_columns.  Used by the full-size parity tests as a probe that touches every element of D (D is symmetric,
 * so D V[s] can be compared with the GPU's matrix times the same vector).  Pins: tests/test_oracle_matrix.py
 * (equals co_dm_cheb times V; unit vectors reproduce the column routine; diagonal H). */
void co_dm_cheb_apply(int n, const double* H, double a, double b, const double* c, int M,
                      int nvec, const double* V, double* out) {
    size_t nn = (size_t)n * n;
    double* X = (double*)malloc(sizeof(double) * nn);
    co_scale(n, H, a, b, X);
    double* wm = (double*)malloc(sizeof(double) * n);
    double* wc = (double*)malloc(sizeof(double) * n);
    double* wn = (double*)malloc(sizeof(double) * n);
    for (int s = 0; s < nvec; ++s) {
        const double* v = V + (size_t)s * n;
        double* o = out + (size_t)s * n;
        for (int i = 0; i < n; ++i) { wm[i] = v[i]; o[i] = (M > 0) ? c[0] * v[i] : 0.0; }
        if (M > 1) {
#pragma omp parallel for schedule(static)
            for (int i = 0; i < n; ++i) {
                double acc = 0.0;
                const double* xi = X + (size_t)i * n;
                for (int kk = 0; kk < n; ++kk) acc += xi[kk] * v[kk];
                wc[i] = acc;
            }
            for (int i = 0; i < n; ++i) o[i] += c[1] * wc[i];
        }
        for (int t = 2; t < M; ++t) {
#pragma omp parallel for schedule(static)
            for (int i = 0; i < n; ++i) {
                double acc = 0.0;
                const double* xi = X + (size_t)i * n;
                for (int kk = 0; kk < n; ++kk) acc += xi[kk] * wc[kk];
                wn[i] = 2.0 * acc - wm[i];
            }
            double* sw = wm; wm = wc; wc = wn; wn = sw;
            for (int i = 0; i < n; ++i) o[i] += c[t] * wc[i];
        }
    }
    free(X); free(wm); free(wc); free(wn);
}

/* Scalar M-term Chebyshev sum by the DEFINITION T_n(x) = cos(n arccos x), |x| <= 1. */
double co_eval_cheb_sum(const double* c, int M, double x) {
    long double th = acosl((long double)x), s = 0.0L;
    for (int n = 0; n < M; ++n) s += (long double)c[n] * cosl((long double)n * th);
    return (double)s;
}

/* ------------------------------------------------------------------------------------------
 * Eq. (9)-(11): T_k^j = sum_l a_{j,l} T_{l k}; recurrence Eq. (10) with
 * a_{0,0}=1, a_{1,0}=0, a_{1,1}=1.  A is p x p row-major, A[j*p+l] = a_{j,l}.
 * ---------------------------------------------------------------------------------------- */
void co_a_matrix(int p, double* A) {
    for (int t = 0; t < p * p; ++t) A[t] = 0.0;
    A[0] = 1.0;
    if (p > 1) { A[1 * p + 0] = 0.0; A[1 * p + 1] = 1.0; }
    for (int j = 2; j < p; ++j) {
        for (int l = 0; l <= j; ++l) {
            double am1 = (l - 1 >= 0 && l - 1 <= j - 1) ? A[(j - 1) * p + (l - 1)] : 0.0;
            double ap1 = (l + 1 <= j - 1) ? A[(j - 1) * p + (l + 1)] : 0.0;
            double v;
            if (l == 0) v = 0.5 * ap1;                                   /* 1/2 a_{j-1,1}            */
            else if (l == 1) v = A[(j - 1) * p + 0] + 0.5 * ap1;         /* a_{j-1,0} + 1/2 a_{j-1,2} */
            else if (l < j) v = 0.5 * (am1 + ap1);
            else v = 0.5 * am1;                                          /* l == j */
            A[j * p + l] = v;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * The km x km system of Eq. (19)-(20), PAPER.md:171-182 (Eq. 20's display is missing from
 * PAPER.md; reconstructed from Eq. 16-17, and the Appendix blocks
 * DESIGN.md reading A4).  Ordering: unknown d_{i,j} sits at
 * index j*k+i, coefficient c_{l k+i} at row l*k+i (Eq. 19's stacking).  K = k*p, Xm is K x K.
 *   row (l, i=0):   c_{lk}   = sum_j a_{j,l} d_{0,j}                                   (Eq. 16)
 *   row (l, i>=1):  c_{lk+i} = w_l sum_j a_{j,l} d_{i,j} + 1/2 sum_j a_{j,l+1} d_{k-i,j} (Eq. 17)
 * with w_0 = 1, w_{l>=1} = 1/2 and a_{j,p} := 0.
 * ---------------------------------------------------------------------------------------- */
void co_x_matrix(int k, int p, const double* A, double* Xm) {
    int K = k * p;
    for (size_t t = 0; t < (size_t)K * K; ++t) Xm[t] = 0.0;
    for (int l = 0; l < p; ++l) {
        for (int j = 0; j < p; ++j) {
            double ajl = A[j * p + l];
            double ajl1 = (l + 1 < p) ? A[j * p + (l + 1)] : 0.0;
            Xm[(size_t)(l * k + 0) * K + (j * k + 0)] += ajl;
            double w = (l == 0) ? 1.0 : 0.5;
            for (int i = 1; i < k; ++i) {
                Xm[(size_t)(l * k + i) * K + (j * k + i)] += w * ajl;          /* I block */
                Xm[(size_t)(l * k + i) * K + (j * k + (k - i))] += 0.5 * ajl1; /* J block */
            }
        }
    }
}

/* Back substitution of an upper-triangular K x K system U x = rhs.  Returns the largest
 * |U[r][c]|, c < r (should be exactly 0 for Eq. 20: "upper-triangular"). */
double co_back_substitute(int K, const double* U, const double* rhs, double* x) {
    double lower = 0.0;
    for (int r = K - 1; r >= 0; --r) {
        long double s = rhs[r];
        for (int cc = r + 1; cc < K; ++cc) s -= (long double)U[(size_t)r * K + cc] * x[cc];
        x[r] = (double)(s / U[(size_t)r * K + r]);
        for (int cc = 0; cc < r; ++cc)
            if (fabs(U[(size_t)r * K + cc]) > lower) lower = fabs(U[(size_t)r * K + cc]);
    }
    return lower;
}

/* Route 1 (the paper's): assemble X (Eq. 20) and back-substitute X d = c.
 * c has k*p entries (zero-padded beyond M by the caller).  d[i*p + j] = d_{i,j}. */
void co_d_from_c_via_X(int k, int p, const double* c, double* d) {
    int K = k * p;
    double* A = (double*)malloc(sizeof(double) * p * p);
    double* Xm = (double*)malloc(sizeof(double) * (size_t)K * K);
    double* sol = (double*)malloc(sizeof(double) * K);
    co_a_matrix(p, A);
    co_x_matrix(k, p, A, Xm);
    co_back_substitute(K, Xm, c, sol);
    for (int j = 0; j < p; ++j)
        for (int i = 0; i < k; ++i) d[i * p + j] = sol[j * k + i];
    free(A); free(Xm); free(sol);
}

/* Route 2: Eq. (16)-(17) solved block by block for g_{i,l} := d_i^T a_l,
 * descending l; g[i*p + l].
 *   g_{0,l}   = c_{lk}
 *   g_{i,p-1} = 2 c_{(p-1)k+i}
 *   g_{i,l}   = 2 c_{lk+i} - g_{k-i,l+1}          1 <= l <= p-2
 *   g_{i,0}   = c_i - 1/2 g_{k-i,1}               (p >= 2);   g_{i,0} = c_i if p == 1
 */
void co_g_from_c(int k, int p, const double* c, double* g) {
    for (int l = 0; l < p; ++l) g[0 * p + l] = c[l * k];
    for (int l = p - 1; l >= 0; --l) {
        for (int i = 1; i < k; ++i) {
            double v;
            if (p == 1) v = c[i];
            else if (l == p - 1) v = 2.0 * c[l * k + i];
            else if (l >= 1) v = 2.0 * c[l * k + i] - g[(k - i) * p + (l + 1)];
            else v = c[i] - 0.5 * g[(k - i) * p + 1];
            g[i * p + l] = v;
        }
    }
}

/* ...then d_i from g_i through Eq. (24): sum_j a_{j,l} d_{i,j} = g_{i,l}
 * (upper-triangular in (l,j) because a_{j,l}=0 for l>j), back substitution per i. */
void co_d_from_g(int k, int p, const double* g, double* d) {
    double* A = (double*)malloc(sizeof(double) * p * p);
    co_a_matrix(p, A);
    for (int i = 0; i < k; ++i) {
        for (int l = p - 1; l >= 0; --l) {
            long double s = g[i * p + l];
            for (int j = l + 1; j < p; ++j) s -= (long double)A[j * p + l] * d[i * p + j];
            d[i * p + l] = (double)(s / A[l * p + l]);
        }
    }
    free(A);
}

/* Scalar right-hand side of Eq. (4), PAPER.md:93 (nested form), with T_i(x) = cos(i arccos x):
 *   acc = S_{p-1};  acc = S_j + T_k * acc,  j = p-2..0;   S_j = sum_{i<k} d_{i,j} T_i.  */
double co_eval_eq4(int k, int p, const double* d, double x) {
    long double th = acosl((long double)x);
    long double Tk = cosl((long double)k * th);
    long double acc = 0.0L;
    for (int j = p - 1; j >= 0; --j) {
        long double S = 0.0L;
        for (int i = 0; i < k; ++i) S += (long double)d[i * p + j] * cosl((long double)i * th);
        acc = S + Tk * acc;
    }
    return (double)acc;
}

/* Scalar right-hand side of Eq. (6): sum_j sum_i d_{i,j} T_k^j T_i. */
double co_eval_eq6(int k, int p, const double* d, double x) {
    long double th = acosl((long double)x);
    long double Tk = cosl((long double)k * th), pw = 1.0L, s = 0.0L;
    for (int j = 0; j < p; ++j) {
        for (int i = 0; i < k; ++i) s += (long double)d[i * p + j] * pw * cosl((long double)i * th);
        pw *= Tk;
    }
    return (double)s;
}

/* ------------------------------------------------------------------------------------------
 * Electron count and chemical potential (north_star item 4; the paper fixes mu = 0,
 * DESIGN.md reading A9):  N_e(mu) = tr sum_n c_n(mu) T_n(X) = sum_n c_n(mu) tau_n
 * with tau_n = tr T_n(X);  mu by bisection on [a,b], exactly `iters` halvings, keeping the
 * invariant N_e(lo) >= N_occ >= N_e(hi) (f is decreasing in eps - mu => N_e increasing in mu,
 * so: if N_e(mid) < N_occ then lo = mid else hi = mid); returns (lo+hi)/2.
 * ---------------------------------------------------------------------------------------- */
double co_electron_count(const double* tau, double beta, double mu, double a, double b, int M, int Nq) {
    double* c = (double*)malloc(sizeof(double) * M);
    co_cheb_coeffs(beta, mu, a, b, M, Nq, c);
    long double s = 0.0L;
    for (int n = 0; n < M; ++n) s += (long double)c[n] * tau[n];
    free(c);
    return (double)s;
}

double co_solve_mu(const double* tau, double beta, double a, double b, int M, int Nq, double n_occ,
                   int iters) {
    double lo = a, hi = b;
    for (int it = 0; it < iters; ++it) {
        double mid = 0.5 * (lo + hi);
        double ne = co_electron_count(tau, beta, mid, a, b, M, Nq);
        if (ne < n_occ) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

/* Exact-spectrum counterpart (for reporting mu_exact): bisection on sum_i f(eps_i). */
double co_solve_mu_exact(int n, const double* E, double beta, double lo, double hi, double n_occ,
                         int iters) {
    for (int it = 0; it < iters; ++it) {
        double mid = 0.5 * (lo + hi), s = 0.0;
        for (int i = 0; i < n; ++i) s += co_fermi(beta, mid, E[i]);
        if (s < n_occ) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}
