/*
 * elpa2_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, CPU-only FP64 oracle for the stage-2 eigenvector back-transformation of the
 * two-stage ELPA2 eigensolver (arxiv 2002.10991, Eq. 6d) and for the step that produces its
 * input (Eq. 6b, bulge chasing).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this library.  It shares no code with the CUDA
 * path (paper_2002_10991_b200/csrc) and must never be called from it.
 *
 * Every function cites the passage of /root/reference/PAPER.md ("PAPER.md:<line>") it follows,
 * or the reading in DESIGN.md ("R<n>") where the paper is silent.  All indices are 0-based:
 * the paper's stage i and sweep j are s = i-1 and k = j-1 here (R1).
 *
 * Parity pins (tests/test_oracle_*.py, "-m 'not gpu'"): nothing here is "parity unpinned".
 *   orc_hh_*            : worked example N=17, b=4 of PAPER.md Figs. 1-4 (tests/golden/)
 *   orc_larfg_*         : H^H x = beta e1, |beta| = ||x||, H^H H = I, Im beta = 0
 *   orc_bulge_chase_*   : dense Q2 gives Q2^H B Q2 = T, Q2^H Q2 = I to 1e-13; eig(T) = eig(B)
 *                         via numpy.linalg.eigvalsh; nbw >= N-1 reduces to one reflector per column
 *   orc_tridiag_ql      : T X = X Lambda, X^T X = I; eigenvalues vs numpy.linalg.eigvalsh
 *   orc_back_transform_*: equals dense Q2 * X; X = I returns Q2; column norms preserved;
 *                         end-to-end ||B Y - Y Lambda|| / ||B|| <= 1e-12 N
 *   orc_full_to_band_* / orc_band_to_full_back_* (Eqs. 6a, 6e): see the block comment above them
 *
 * Build: gcc -O2 -std=c99 -fopenmp -shared -fPIC -o libelpa2_oracle.so elpa2_oracle.c -lm
 * (no -ffast-math; OpenMP is used only to spread independent eigenvector columns,
 * PAPER.md:134, over the host cores in orc_back_transform_*).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex zdouble;

/* ------------------------------------------------------------------------------------------
 * Reflector layout (R3, R4; "N-2 stages, (N-i)/b sweeps in the i-th
 * stage", "Most Householder vectors have a length equal to b, except that
 * [those] generated in the last sweep of each stage may be shorter").
 *
 * Sweep s = 0..N-2 has K(s) = ceil((N-1-s)/nbw) chase blocks k = 0..K(s)-1.  Reflector (s,k)
 * acts on rows r0 = s+1+k*nbw .. r1 = min(s+(k+1)*nbw, N-1).  Slots are numbered in generation
 * order (s outer, k inner).  Written as plain sums on purpose (the CUDA library uses a closed
 * form; tests compare the two).
 * ---------------------------------------------------------------------------------------- */
int orc_hh_blocks(int64_t N, int nbw, int64_t s)
{
    if (N < 2 || nbw < 1 || s < 0 || s > N - 2) return 0;
    int64_t rows = N - 1 - s;              /* rows below the diagonal in column s */
    return (int)((rows + nbw - 1) / nbw);
}

int64_t orc_hh_offset(int64_t N, int nbw, int64_t s)
{
    int64_t off = 0;
    for (int64_t t = 0; t < s && t <= N - 2; ++t) off += orc_hh_blocks(N, nbw, t);
    return off;
}

int64_t orc_hh_count(int64_t N, int nbw)
{
    if (N < 2) return 0;
    return orc_hh_offset(N, nbw, N - 1);
}

/* first and last row touched by reflector (s,k); returns its length L */
int orc_hh_rows(int64_t N, int nbw, int64_t s, int k, int64_t *r0, int64_t *r1)
{
    *r0 = s + 1 + (int64_t)k * nbw;
    *r1 = s + ((int64_t)k + 1) * nbw;
    if (*r1 > N - 1) *r1 = N - 1;
    return (int)(*r1 - *r0 + 1);
}

/* ------------------------------------------------------------------------------------------
 * Householder generator ("computed following the standard Householder method";
 * Eq. 7; R2, R7).  Input x[0..L-1] (x[0] = alpha).  Output v (v[0] = 1,
 * length L), tau, beta (real) such that H^H x = beta e1 with H = I - tau v v^H.
 *   sigma = ||x[1:]||;  if sigma = 0 and Im alpha = 0: tau = 0, v = e1, beta = alpha
 *   else beta = -sign(Re alpha) sqrt(|alpha|^2 + sigma^2), sign(0) = +1
 *        tau = (beta - alpha)/beta;  v[i] = x[i]/(alpha - beta)
 * ---------------------------------------------------------------------------------------- */
void orc_larfg_d(int L, const double *x, double *v, double *tau, double *beta)
{
    double alpha = x[0], ss = 0.0;
    for (int i = 1; i < L; ++i) ss += x[i] * x[i];
    v[0] = 1.0;
    if (ss == 0.0) {
        for (int i = 1; i < L; ++i) v[i] = 0.0;
        *tau = 0.0;
        *beta = alpha;
        return;
    }
    double nrm = sqrt(alpha * alpha + ss);
    double b = (alpha >= 0.0) ? -nrm : nrm;
    *tau = (b - alpha) / b;
    double scal = 1.0 / (alpha - b);
    for (int i = 1; i < L; ++i) v[i] = x[i] * scal;
    *beta = b;
}

void orc_larfg_z(int L, const zdouble *x, zdouble *v, zdouble *tau, double *beta)
{
    zdouble alpha = x[0];
    double ar = creal(alpha), ai = cimag(alpha), ss = 0.0;
    for (int i = 1; i < L; ++i) ss += creal(x[i]) * creal(x[i]) + cimag(x[i]) * cimag(x[i]);
    v[0] = 1.0;
    if (ss == 0.0 && ai == 0.0) {
        for (int i = 1; i < L; ++i) v[i] = 0.0;
        *tau = 0.0;
        *beta = ar;
        return;
    }
    double nrm = sqrt(ar * ar + ai * ai + ss);
    double b = (ar >= 0.0) ? -nrm : nrm;
    *tau = ((b - ar) / b) + (-ai / b) * I;
    zdouble scal = 1.0 / (alpha - b);
    for (int i = 1; i < L; ++i) v[i] = x[i] * scal;
    *beta = b;
}

/* ------------------------------------------------------------------------------------------
 * Band -> tridiagonal by bulge chasing (Eq. 6b; Fig. 2), emitting
 * the reflectors of Eq. 7 into a separate array.  DESIGN.md R2-R5.
 *
 * Storage: lower band with 2*nbw sub-diagonals (the fill reaches distance 2*nbw-1):
 *   B[i][j], 0 <= i-j <= 2*nbw, at ab[(i-j) + j*(2*nbw+1)].  On entry everything at distance
 *   > nbw is zero.  On exit ab holds T (plus zeros).
 *
 * For s = 0..N-2 ("stage"), k = 0..K(s)-1 ("sweep"): rows R = r0..r1; the column to clear is
 * c = s for k = 0 ("The first sweep of the i-th stage reduces the i-th column")
 * and c = r0-nbw for k >= 1 ("the first column of the fill-ins introduced in the previous
 * sweep is eliminated").  (v, tau, beta) = larfg(B[R][c]); B <- H^H B H touches
 *   (i)   A = B[R][c+1 .. r0-1]        <- H^H A      (rest of the bulge block; empty for k = 0)
 *   (ii)  D = B[R][R]                  <- H^H D H    (Hermitian)
 *   (iii) E = B[r1+1 .. min(r1+nbw,N-1)][R] <- E H   (creates the next bulge)
 * A length-1 "reflector" with k >= 1 has nothing to eliminate and is stored as identity.
 * v is stored zero-padded to nbw with v[0] = 1 (R8).
 * d[0..N-1], e[0..N-2] receive the tridiagonal (e real by construction, R4).
 * ---------------------------------------------------------------------------------------- */
#define BD(i, j) ab[((i) - (j)) + (j) * ldab]

int orc_bulge_chase_d(int64_t N, int nbw, double *ab, double *hh_v, double *hh_tau,
                      double *d, double *e)
{
    const int64_t ldab = 2 * (int64_t)nbw + 1;
    double *x = malloc(sizeof(double) * nbw), *v = malloc(sizeof(double) * nbw);
    double *w = malloc(sizeof(double) * nbw);
    double *D = malloc(sizeof(double) * nbw * nbw), *M = malloc(sizeof(double) * nbw * nbw);
    if (!x || !v || !w || !D || !M) return -1;
    int64_t g = 0;
    for (int64_t s = 0; s + 2 <= N; ++s) {
        int K = orc_hh_blocks(N, nbw, s);
        for (int k = 0; k < K; ++k, ++g) {
            int64_t r0, r1;
            int L = orc_hh_rows(N, nbw, s, k, &r0, &r1);
            int64_t c = (k == 0) ? s : r0 - nbw;
            double *vout = hh_v + g * nbw;
            for (int i = 0; i < nbw; ++i) vout[i] = 0.0;
            vout[0] = 1.0;
            hh_tau[g] = 0.0;
            if (k > 0 && L == 1) continue;
            double tau, beta;
            for (int i = 0; i < L; ++i) x[i] = BD(r0 + i, c);
            orc_larfg_d(L, x, v, &tau, &beta);
            for (int i = 0; i < L; ++i) vout[i] = v[i];
            hh_tau[g] = tau;
            BD(r0, c) = beta;
            for (int i = 1; i < L; ++i) BD(r0 + i, c) = 0.0;
            if (tau == 0.0) continue;
            /* (i) A <- H^H A = A - tau v (v^T A) */
            for (int64_t j = c + 1; j < r0; ++j) {
                double dot = 0.0;
                for (int i = 0; i < L; ++i) dot += v[i] * BD(r0 + i, j);
                for (int i = 0; i < L; ++i) BD(r0 + i, j) -= tau * v[i] * dot;
            }
            /* (ii) D <- H^H D H on the full symmetric L x L block */
            for (int j = 0; j < L; ++j)
                for (int i = 0; i < L; ++i)
                    D[i + j * L] = (i >= j) ? BD(r0 + i, r0 + j) : BD(r0 + j, r0 + i);
            for (int j = 0; j < L; ++j) {        /* M = D - tau v (v^T D) */
                double dot = 0.0;
                for (int i = 0; i < L; ++i) dot += v[i] * D[i + j * L];
                w[j] = dot;
            }
            for (int j = 0; j < L; ++j)
                for (int i = 0; i < L; ++i) M[i + j * L] = D[i + j * L] - tau * v[i] * w[j];
            for (int i = 0; i < L; ++i) {        /* w = M v */
                double dot = 0.0;
                for (int j = 0; j < L; ++j) dot += M[i + j * L] * v[j];
                w[i] = dot;
            }
            for (int j = 0; j < L; ++j)          /* D' = M - tau (M v) v^T, lower part kept */
                for (int i = j; i < L; ++i) BD(r0 + i, r0 + j) = M[i + j * L] - tau * w[i] * v[j];
            /* (iii) E <- E H = E - tau (E v) v^T */
            int64_t r2 = r1 + nbw;
            if (r2 > N - 1) r2 = N - 1;
            for (int64_t i = r1 + 1; i <= r2; ++i) {
                double dot = 0.0;
                for (int l = 0; l < L; ++l) dot += BD(i, r0 + l) * v[l];
                for (int l = 0; l < L; ++l) BD(i, r0 + l) -= tau * dot * v[l];
            }
        }
    }
    for (int64_t i = 0; i < N; ++i) d[i] = BD(i, i);
    for (int64_t i = 0; i + 1 < N; ++i) e[i] = BD(i + 1, i);
    free(x); free(v); free(w); free(D); free(M);
    return 0;
}
#undef BD

#define BZ(i, j) ab[((i) - (j)) + (j) * ldab]

/* Complex Hermitian version.  Complex tau convention (R2): generation applies
 * B <- H^H B H with H = I - tau v v^H, H^H = I - conj(tau) v v^H. */
int orc_bulge_chase_z(int64_t N, int nbw, zdouble *ab, zdouble *hh_v, zdouble *hh_tau,
                      double *d, double *e)
{
    const int64_t ldab = 2 * (int64_t)nbw + 1;
    zdouble *x = malloc(sizeof(zdouble) * nbw), *v = malloc(sizeof(zdouble) * nbw);
    zdouble *w = malloc(sizeof(zdouble) * nbw);
    zdouble *D = malloc(sizeof(zdouble) * nbw * nbw), *M = malloc(sizeof(zdouble) * nbw * nbw);
    if (!x || !v || !w || !D || !M) return -1;
    int64_t g = 0;
    for (int64_t s = 0; s + 2 <= N; ++s) {
        int K = orc_hh_blocks(N, nbw, s);
        for (int k = 0; k < K; ++k, ++g) {
            int64_t r0, r1;
            int L = orc_hh_rows(N, nbw, s, k, &r0, &r1);
            int64_t c = (k == 0) ? s : r0 - nbw;
            zdouble *vout = hh_v + g * nbw;
            for (int i = 0; i < nbw; ++i) vout[i] = 0.0;
            vout[0] = 1.0;
            hh_tau[g] = 0.0;
            if (k > 0 && L == 1) continue;
            zdouble tau;
            double beta;
            for (int i = 0; i < L; ++i) x[i] = BZ(r0 + i, c);
            orc_larfg_z(L, x, v, &tau, &beta);
            for (int i = 0; i < L; ++i) vout[i] = v[i];
            hh_tau[g] = tau;
            BZ(r0, c) = beta;
            for (int i = 1; i < L; ++i) BZ(r0 + i, c) = 0.0;
            if (tau == 0.0) continue;
            zdouble ctau = conj(tau);
            /* (i) A <- H^H A = A - conj(tau) v (v^H A) */
            for (int64_t j = c + 1; j < r0; ++j) {
                zdouble dot = 0.0;
                for (int i = 0; i < L; ++i) dot += conj(v[i]) * BZ(r0 + i, j);
                for (int i = 0; i < L; ++i) BZ(r0 + i, j) -= ctau * v[i] * dot;
            }
            /* (ii) D <- H^H D H on the full Hermitian L x L block */
            for (int j = 0; j < L; ++j)
                for (int i = 0; i < L; ++i)
                    D[i + j * L] = (i >= j) ? BZ(r0 + i, r0 + j) : conj(BZ(r0 + j, r0 + i));
            for (int j = 0; j < L; ++j) {        /* M = D - conj(tau) v (v^H D) */
                zdouble dot = 0.0;
                for (int i = 0; i < L; ++i) dot += conj(v[i]) * D[i + j * L];
                w[j] = dot;
            }
            for (int j = 0; j < L; ++j)
                for (int i = 0; i < L; ++i) M[i + j * L] = D[i + j * L] - ctau * v[i] * w[j];
            for (int i = 0; i < L; ++i) {        /* w = M v */
                zdouble dot = 0.0;
                for (int j = 0; j < L; ++j) dot += M[i + j * L] * v[j];
                w[i] = dot;
            }
            for (int j = 0; j < L; ++j)          /* D' = M - tau (M v) v^H, lower part kept */
                for (int i = j; i < L; ++i)
                    BZ(r0 + i, r0 + j) = M[i + j * L] - tau * w[i] * conj(v[j]);
            for (int i = 0; i < L; ++i)          /* a Hermitian diagonal is real */
                BZ(r0 + i, r0 + i) = creal(BZ(r0 + i, r0 + i));
            /* (iii) E <- E H = E - tau (E v) v^H */
            int64_t r2 = r1 + nbw;
            if (r2 > N - 1) r2 = N - 1;
            for (int64_t i = r1 + 1; i <= r2; ++i) {
                zdouble dot = 0.0;
                for (int l = 0; l < L; ++l) dot += BZ(i, r0 + l) * v[l];
                for (int l = 0; l < L; ++l) BZ(i, r0 + l) -= tau * dot * conj(v[l]);
            }
        }
    }
    for (int64_t i = 0; i < N; ++i) d[i] = creal(BZ(i, i));
    for (int64_t i = 0; i + 1 < N; ++i) e[i] = creal(BZ(i + 1, i));
    free(x); free(v); free(w); free(D); free(M);
    return 0;
}
#undef BZ

/* ------------------------------------------------------------------------------------------
 * Tridiagonal eigenpairs (Eq. 6c; used only to make X for configs 1-2).  The paper
 * uses divide-and-conquer; BASELINE.json prescribes the textbook implicit-shift
 * QL iteration with Wilkinson shift of the paper's Ref. [11] (R9).
 * In: d[0..N-1], e[0..N-2] (destroyed).  Out: d = eigenvalues ascending; x (N x N, column-major,
 * ldx = N) = eigenvectors as columns.  Returns 0, or l+1 if eigenvalue l did not converge.
 * ---------------------------------------------------------------------------------------- */
int orc_tridiag_ql(int64_t N, double *d, double *e_in, double *x)
{
    const int64_t n = N;
    double *e = malloc(sizeof(double) * (n > 0 ? n : 1));
    if (!e) return -1;
    for (int64_t i = 0; i + 1 < n; ++i) e[i] = e_in[i];
    if (n > 0) e[n - 1] = 0.0;
    for (int64_t j = 0; j < n; ++j)
        for (int64_t i = 0; i < n; ++i) x[i + j * n] = (i == j) ? 1.0 : 0.0;
    const double eps = 2.220446049250313e-16;
    for (int64_t l = 0; l < n; ++l) {
        int iter = 0;
        int64_t m;
        do {
            for (m = l; m + 1 < n; ++m) {           /* look for a negligible sub-diagonal */
                double dd = fabs(d[m]) + fabs(d[m + 1]);
                if (fabs(e[m]) <= eps * dd) break;
            }
            if (m != l) {
                if (iter++ == 200) { free(e); return (int)(l + 1); }
                double g = (d[l + 1] - d[l]) / (2.0 * e[l]);      /* Wilkinson shift */
                double r = hypot(g, 1.0);
                g = d[m] - d[l] + e[l] / (g + (g >= 0.0 ? fabs(r) : -fabs(r)));
                double sn = 1.0, cs = 1.0, p = 0.0;
                int64_t i;
                for (i = m - 1; i >= l; --i) {      /* plane rotations chase the bulge up */
                    double f = sn * e[i], b = cs * e[i];
                    r = hypot(f, g);
                    e[i + 1] = r;
                    if (r == 0.0) { d[i + 1] -= p; e[m] = 0.0; break; }
                    sn = f / r;
                    cs = g / r;
                    g = d[i + 1] - p;
                    r = (d[i] - g) * sn + 2.0 * cs * b;
                    p = sn * r;
                    d[i + 1] = g + p;
                    g = cs * r - b;
                    double *xi = x + i * n, *xi1 = x + (i + 1) * n;   /* accumulate into X */
                    for (int64_t t = 0; t < n; ++t) {
                        double fz = xi1[t];
                        xi1[t] = sn * xi[t] + cs * fz;
                        xi[t] = cs * xi[t] - sn * fz;
                    }
                }
                if (r == 0.0 && i >= l) continue;
                d[l] -= p;
                e[l] = g;
                e[m] = 0.0;
            }
        } while (m != l);
    }
    free(e);
    /* selection sort ascending, permuting the columns of X with the eigenvalues */
    for (int64_t i = 0; i + 1 < n; ++i) {
        int64_t kmin = i;
        for (int64_t j = i + 1; j < n; ++j) if (d[j] < d[kmin]) kmin = j;
        if (kmin != i) {
            double t = d[i]; d[i] = d[kmin]; d[kmin] = t;
            for (int64_t r = 0; r < n; ++r) {
                double tt = x[r + i * n]; x[r + i * n] = x[r + kmin * n]; x[r + kmin * n] = tt;
            }
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * The back-transformation itself (Eq. 6d; Eq. 8): apply every
 * H(s,k) = I - tau v v^H to q, the reflector generated last first ("the reverse of the order in
 * which they are generated").  This is the plain definition:
 *
 *   for s = N-2 .. 0:  for k = 0 .. K(s)-1:   (all reflectors of one sweep act on disjoint rows)
 *       for each column x of q:  d = sum_r conj(v[r]) x[r0+r];   x[r0+r] -= tau * d * v[r]
 *
 * tau is used as stored, NOT conjugated (R2).  q is column-major N x ncols with
 * leading dimension ldq, updated in place.  Columns are independent, so the
 * column range is split over OpenMP threads; each thread runs the full reflector loop on its
 * own columns in exactly the order above.
 * ---------------------------------------------------------------------------------------- */
/* Columns handed to one thread at a time: up to 8 (they share each reflector while it is in
 * cache), fewer when there are not enough columns to give every thread a chunk.  Scheduling only:
 * each column sees exactly the same operations in the same order whatever the chunk size. */
static int64_t orc_col_chunk(int64_t ncols)
{
    int64_t nt = 1;
#ifdef _OPENMP
    nt = omp_get_max_threads();
#endif
    int64_t c = (ncols + nt - 1) / nt;
    if (c > 8) c = 8;
    if (c < 1) c = 1;
    return c;
}

void orc_back_transform_d(int64_t N, int nbw, int64_t ncols, const double *hh_v,
                          const double *hh_tau, double *q, int64_t ldq)
{
    if (N < 2 || ncols < 1) return;
    int64_t *off = malloc(sizeof(int64_t) * N);
    off[0] = 0;
    for (int64_t s = 1; s < N; ++s) off[s] = off[s - 1] + orc_hh_blocks(N, nbw, s - 1);
    const int64_t chunk = orc_col_chunk(ncols);
    const int64_t nchunks = (ncols + chunk - 1) / chunk;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t cb = 0; cb < nchunks; ++cb) {
        int64_t j0 = cb * chunk, j1 = j0 + chunk < ncols ? j0 + chunk : ncols;
        for (int64_t s = N - 2; s >= 0; --s) {
            int K = orc_hh_blocks(N, nbw, s);
            for (int k = 0; k < K; ++k) {
                int64_t g = off[s] + k, r0, r1;
                int L = orc_hh_rows(N, nbw, s, k, &r0, &r1);
                double tau = hh_tau[g];
                if (tau == 0.0) continue;
                const double *v = hh_v + g * nbw;
                for (int64_t j = j0; j < j1; ++j) {
                    double *x = q + r0 + j * ldq;
                    double dot = 0.0;
                    for (int r = 0; r < L; ++r) dot += v[r] * x[r];
                    double td = tau * dot;
                    for (int r = 0; r < L; ++r) x[r] -= td * v[r];
                }
            }
        }
    }
    free(off);
}

void orc_back_transform_z(int64_t N, int nbw, int64_t ncols, const zdouble *hh_v,
                          const zdouble *hh_tau, zdouble *q, int64_t ldq)
{
    if (N < 2 || ncols < 1) return;
    int64_t *off = malloc(sizeof(int64_t) * N);
    off[0] = 0;
    for (int64_t s = 1; s < N; ++s) off[s] = off[s - 1] + orc_hh_blocks(N, nbw, s - 1);
    const int64_t chunk = orc_col_chunk(ncols);
    const int64_t nchunks = (ncols + chunk - 1) / chunk;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t cb = 0; cb < nchunks; ++cb) {
        int64_t j0 = cb * chunk, j1 = j0 + chunk < ncols ? j0 + chunk : ncols;
        for (int64_t s = N - 2; s >= 0; --s) {
            int K = orc_hh_blocks(N, nbw, s);
            for (int k = 0; k < K; ++k) {
                int64_t g = off[s] + k, r0, r1;
                int L = orc_hh_rows(N, nbw, s, k, &r0, &r1);
                zdouble tau = hh_tau[g];
                if (tau == 0.0) continue;
                const zdouble *v = hh_v + g * nbw;
                for (int64_t j = j0; j < j1; ++j) {
                    zdouble *x = q + r0 + j * ldq;
                    zdouble dot = 0.0;
                    for (int r = 0; r < L; ++r) dot += conj(v[r]) * x[r];
                    zdouble td = tau * dot;
                    for (int r = 0; r < L; ++r) x[r] -= td * v[r];
                }
            }
        }
    }
    free(off);
}

/* ------------------------------------------------------------------------------------------
 * the same definition (Eq. 8 in reverse generation order) in FP32, real and
 * complex (R16: the paper runs ELPA in double precision only; single precision is the
 * library's other build, so the reading is "the same operations with every product and sum rounded
 * to float").  Inputs are the FP64 reflectors rounded to float by the caller.  ISO C, no FMA
 * contraction, FLT_EVAL_METHOD 0 on x86-64: each operation is a correctly rounded float operation.
 * Pins (tests/test_oracle_backtransform.py): agrees with orc_back_transform_d/z on the same rounded
 * inputs to the FP32 error bound of DESIGN.md "Tolerance (FP32)", preserves column norms to that
 * bound, and a reversed order misses it by O(1).
 * ------------------------------------------------------------------------------------------ */
typedef float _Complex zfloat;

void orc_back_transform_s(int64_t N, int nbw, int64_t ncols, const float *hh_v, const float *hh_tau,
                          float *q, int64_t ldq)
{
    if (N < 2 || ncols < 1) return;
    int64_t *off = malloc(sizeof(int64_t) * N);
    off[0] = 0;
    for (int64_t s = 1; s < N; ++s) off[s] = off[s - 1] + orc_hh_blocks(N, nbw, s - 1);
    const int64_t chunk = orc_col_chunk(ncols);
    const int64_t nchunks = (ncols + chunk - 1) / chunk;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t cb = 0; cb < nchunks; ++cb) {
        int64_t j0 = cb * chunk, j1 = j0 + chunk < ncols ? j0 + chunk : ncols;
        for (int64_t s = N - 2; s >= 0; --s) {
            int K = orc_hh_blocks(N, nbw, s);
            for (int k = 0; k < K; ++k) {
                int64_t g = off[s] + k, r0, r1;
                int L = orc_hh_rows(N, nbw, s, k, &r0, &r1);
                float tau = hh_tau[g];
                if (tau == 0.0f) continue;
                const float *v = hh_v + g * nbw;
                for (int64_t j = j0; j < j1; ++j) {
                    float *x = q + r0 + j * ldq;
                    float dot = 0.0f;
                    for (int r = 0; r < L; ++r) dot += v[r] * x[r];
                    float td = tau * dot;
                    for (int r = 0; r < L; ++r) x[r] -= td * v[r];
                }
            }
        }
    }
    free(off);
}

void orc_back_transform_c(int64_t N, int nbw, int64_t ncols, const zfloat *hh_v, const zfloat *hh_tau,
                          zfloat *q, int64_t ldq)
{
    if (N < 2 || ncols < 1) return;
    int64_t *off = malloc(sizeof(int64_t) * N);
    off[0] = 0;
    for (int64_t s = 1; s < N; ++s) off[s] = off[s - 1] + orc_hh_blocks(N, nbw, s - 1);
    const int64_t chunk = orc_col_chunk(ncols);
    const int64_t nchunks = (ncols + chunk - 1) / chunk;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t cb = 0; cb < nchunks; ++cb) {
        int64_t j0 = cb * chunk, j1 = j0 + chunk < ncols ? j0 + chunk : ncols;
        for (int64_t s = N - 2; s >= 0; --s) {
            int K = orc_hh_blocks(N, nbw, s);
            for (int k = 0; k < K; ++k) {
                int64_t g = off[s] + k, r0, r1;
                int L = orc_hh_rows(N, nbw, s, k, &r0, &r1);
                zfloat tau = hh_tau[g];
                if (tau == 0.0f) continue;
                const zfloat *v = hh_v + g * nbw;
                for (int64_t j = j0; j < j1; ++j) {
                    zfloat *x = q + r0 + j * ldq;
                    zfloat dot = 0.0f;
                    for (int r = 0; r < L; ++r) dot += conjf(v[r]) * x[r];
                    zfloat td = tau * dot;
                    for (int r = 0; r < L; ++r) x[r] -= td * v[r];
                }
            }
        }
    }
    free(off);
}

int orc_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        n = omp_get_num_threads();
    }
#endif
    return n;
}

/* ==========================================================================================
 * the steps around the band stage -- full -> band (Eq. 6a, PAPER.md:84:
 * B = P H P*) and the band -> full back-transformation of the eigenvectors (Eq. 6e, PAPER.md:93:
 * C = P* Y).  The paper gives the two equations and says 6a "mostly involves ... BLAS level-3
 * matrix-matrix operations", nothing else; the reading taken here is DESIGN.md R15:
 *
 *   P* = H_0 H_1 ... H_{Nv-1},  Nv = max(N - nbw - 1, 0),  H_j = I - tau_j v_j v_j^H  (Eq. 7's form,
 *   PAPER.md:121, with the larfg convention of R2/R7), where reflector j clears column j below the
 *   band: it acts on rows j+nbw .. N-1 and is generated from H^(j)[j+nbw .. N-1][j], H^(j) being the
 *   matrix after the first j two-sided updates  H <- H_j^H H H_j.
 *
 * A blocked (panel QR + trailing update) reduction produces the same reflectors up to rounding: the
 * right-hand applications of H_j touch columns >= j+nbw only, i.e. never the other columns of the
 * panel j belongs to, so deferring them changes nothing.  The oracle is therefore the plain unblocked
 * definition, one reflector at a time on the full matrix, O(N^3): for tests at N <= ~1500.
 *
 * Reflector storage (the layout elpa2_trans_ev_band_to_full_* consumes, include/elpa2_bt.h):
 *   hv: column-major N x Nv, leading dimension ldv >= N; column j holds v_j at rows j+nbw .. N-1
 *   with hv[j+nbw + j*ldv] == 1 stored explicitly and rows < j+nbw ZERO;  tau[j], j < Nv.
 *
 * Pins (tests/test_oracle_full.py): dense Qf = H_0 .. H_{Nv-1} from textbook reflectors built in
 * numpy gives Qf^H H Qf = B (band of semi-bandwidth nbw) and Qf^H Qf = I to 1e-13; eig(B) = eig(H);
 * nbw = 1 equals LAPACK's one-stage tridiagonalization (scipy.linalg.hessenberg); nbw >= N-1 leaves H
 * alone; back-transform = dense Qf * Y, Y = I returns Qf, column norms preserved, and end to end
 * through 6a -> 6b -> 6c -> 6d -> 6e: || H C - C Lambda || / || H || <= 1e-12 N.
 * ========================================================================================== */

/* Eq. 6a.  a: N x N column-major (lda), full Hermitian storage (both triangles), overwritten with
 * the band matrix B (both triangles; entries outside the band are set to exact zeros). */
int orc_full_to_band_d(int64_t N, int nbw, double *a, int64_t lda, double *hv, int64_t ldv, double *tau)
{
    if (N < 0 || nbw < 1 || lda < (N > 1 ? N : 1)) return -1;
    const int64_t Nv = (N - nbw - 1 > 0) ? N - nbw - 1 : 0;
    double *x = malloc(sizeof(double) * (N > 0 ? N : 1)), *v = malloc(sizeof(double) * (N > 0 ? N : 1));
    if (!x || !v) return -2;
    for (int64_t j = 0; j < Nv; ++j) {
        const int64_t r0 = j + nbw;
        const int L = (int)(N - r0);
        double t, beta;
        for (int i = 0; i < L; ++i) x[i] = a[(r0 + i) + j * lda];
        orc_larfg_d(L, x, v, &t, &beta);
        for (int64_t i = 0; i < N; ++i) hv[i + j * ldv] = 0.0;
        for (int i = 0; i < L; ++i) hv[(r0 + i) + j * ldv] = v[i];
        tau[j] = t;
        if (t != 0.0) {
            /* A <- H^T A: rows r0.., every column */
            for (int64_t c = 0; c < N; ++c) {
                double dot = 0.0;
                for (int i = 0; i < L; ++i) dot += v[i] * a[(r0 + i) + c * lda];
                for (int i = 0; i < L; ++i) a[(r0 + i) + c * lda] -= t * v[i] * dot;
            }
            /* A <- A H: columns r0.., every row */
            for (int64_t r = 0; r < N; ++r) {
                double dot = 0.0;
                for (int i = 0; i < L; ++i) dot += a[r + (r0 + i) * lda] * v[i];
                for (int i = 0; i < L; ++i) a[r + (r0 + i) * lda] -= t * dot * v[i];
            }
        }
        /* the eliminated entries are zero by construction, the head is beta */
        a[r0 + j * lda] = beta;
        a[j + r0 * lda] = beta;
        for (int i = 1; i < L; ++i) {
            a[(r0 + i) + j * lda] = 0.0;
            a[j + (r0 + i) * lda] = 0.0;
        }
    }
    free(x); free(v);
    return 0;
}

int orc_full_to_band_z(int64_t N, int nbw, zdouble *a, int64_t lda, zdouble *hv, int64_t ldv, zdouble *tau)
{
    if (N < 0 || nbw < 1 || lda < (N > 1 ? N : 1)) return -1;
    const int64_t Nv = (N - nbw - 1 > 0) ? N - nbw - 1 : 0;
    zdouble *x = malloc(sizeof(zdouble) * (N > 0 ? N : 1)), *v = malloc(sizeof(zdouble) * (N > 0 ? N : 1));
    if (!x || !v) return -2;
    for (int64_t j = 0; j < Nv; ++j) {
        const int64_t r0 = j + nbw;
        const int L = (int)(N - r0);
        zdouble t;
        double beta;
        for (int i = 0; i < L; ++i) x[i] = a[(r0 + i) + j * lda];
        orc_larfg_z(L, x, v, &t, &beta);
        for (int64_t i = 0; i < N; ++i) hv[i + j * ldv] = 0.0;
        for (int i = 0; i < L; ++i) hv[(r0 + i) + j * ldv] = v[i];
        tau[j] = t;
        if (t != 0.0) {
            const zdouble ct = conj(t);
            /* A <- H^H A = A - conj(tau) v (v^H A) */
            for (int64_t c = 0; c < N; ++c) {
                zdouble dot = 0.0;
                for (int i = 0; i < L; ++i) dot += conj(v[i]) * a[(r0 + i) + c * lda];
                for (int i = 0; i < L; ++i) a[(r0 + i) + c * lda] -= ct * v[i] * dot;
            }
            /* A <- A H = A - tau (A v) v^H */
            for (int64_t r = 0; r < N; ++r) {
                zdouble dot = 0.0;
                for (int i = 0; i < L; ++i) dot += a[r + (r0 + i) * lda] * v[i];
                for (int i = 0; i < L; ++i) a[r + (r0 + i) * lda] -= t * dot * conj(v[i]);
            }
        }
        a[r0 + j * lda] = beta;
        a[j + r0 * lda] = beta;
        for (int i = 1; i < L; ++i) {
            a[(r0 + i) + j * lda] = 0.0;
            a[j + (r0 + i) * lda] = 0.0;
        }
    }
    for (int64_t i = 0; i < N; ++i) a[i + i * lda] = creal(a[i + i * lda]);   /* a Hermitian diagonal is real */
    free(x); free(v);
    return 0;
}

/* Eq. 6e: q <- P* q = H_0 (H_1 ( ... (H_{Nv-1} q))), the plain definition: the reflector generated
 * last is applied first, each as x <- x - tau (v^H x) v on rows j+nbw .. N-1 (Eq. 8's form,
 * PAPER.md:162; tau as stored, R2).  Columns are independent: OpenMP over column
 * chunks, each thread running the whole reflector loop on its columns in exactly this order. */
void orc_band_to_full_back_d(int64_t N, int nbw, int64_t ncols, const double *hv, int64_t ldv,
                             const double *tau, double *q, int64_t ldq)
{
    const int64_t Nv = (N - nbw - 1 > 0) ? N - nbw - 1 : 0;
    if (Nv == 0 || ncols < 1) return;
    const int64_t chunk = orc_col_chunk(ncols);
    const int64_t nchunks = (ncols + chunk - 1) / chunk;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t cb = 0; cb < nchunks; ++cb) {
        int64_t j0 = cb * chunk, j1 = j0 + chunk < ncols ? j0 + chunk : ncols;
        for (int64_t j = Nv - 1; j >= 0; --j) {
            const double t = tau[j];
            if (t == 0.0) continue;
            const int64_t r0 = j + nbw, L = N - r0;
            const double *v = hv + r0 + j * ldv;
            for (int64_t c = j0; c < j1; ++c) {
                double *x = q + r0 + c * ldq;
                double dot = 0.0;
                for (int64_t r = 0; r < L; ++r) dot += v[r] * x[r];
                double td = t * dot;
                for (int64_t r = 0; r < L; ++r) x[r] -= td * v[r];
            }
        }
    }
}

void orc_band_to_full_back_z(int64_t N, int nbw, int64_t ncols, const zdouble *hv, int64_t ldv,
                             const zdouble *tau, zdouble *q, int64_t ldq)
{
    const int64_t Nv = (N - nbw - 1 > 0) ? N - nbw - 1 : 0;
    if (Nv == 0 || ncols < 1) return;
    const int64_t chunk = orc_col_chunk(ncols);
    const int64_t nchunks = (ncols + chunk - 1) / chunk;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t cb = 0; cb < nchunks; ++cb) {
        int64_t j0 = cb * chunk, j1 = j0 + chunk < ncols ? j0 + chunk : ncols;
        for (int64_t j = Nv - 1; j >= 0; --j) {
            const zdouble t = tau[j];
            if (t == 0.0) continue;
            const int64_t r0 = j + nbw, L = N - r0;
            const zdouble *v = hv + r0 + j * ldv;
            for (int64_t c = j0; c < j1; ++c) {
                zdouble *x = q + r0 + c * ldq;
                zdouble dot = 0.0;
                for (int64_t r = 0; r < L; ++r) dot += conj(v[r]) * x[r];
                zdouble td = t * dot;
                for (int64_t r = 0; r < L; ++r) x[r] -= td * v[r];
            }
        }
    }
}
