/*
 * submatrix_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, fp64 CPU statement of the submatrix method for the matrix sign
 * function, written from /root/reference/PAPER.md.  It exists to check the CUDA
 * path; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.  It shares no code with the CUDA path.
 *
 * What it follows:
 *   step 1  PAPER.md:110 (Fig. 2)  "construction of a submatrix T_i(A) for every
 *           column of the matrix A"            -> orc_build_pattern, orc_gather
 *   step 2  PAPER.md:110 "the matrix function is applied to the dense
 *           submatrices, f(T_i(A))", with f = sign, Eq. 13
 *           sign(A) = A (A^2)^(-1/2).  For symmetric T = V diag(w) V^T this is,
 *           by definition, V diag(sgn w) V^T; V, w from a cyclic Jacobi
 *           eigendecomposition written out below       -> orc_jacobi, orc_sign
 *   step 3  PAPER.md:110 "the relevant result columns are inserted into the
 *           sparse result matrix"                      -> orc_density_columns
 *   Eq. 14  PAPER.md:91 with S = I: D = 1/2 (I - sign(H - mu I)).
 *
 * Readings where the paper is silent are listed in DESIGN.md section 3 (A1..A19):
 * one submatrix per BLOCK column (A1); the index set of T_i is N(i) = block rows
 * with a stored block in column i, ascending, absent pairs are zero (A2, A3);
 * "relevant columns" = the b_i columns at the local position of block i (A4);
 * sgn(0) := 0 (A14).
 *
 * The second function of the eigendecomposition, the "NS-k polynomial"
 * V diag(g^k(w/s)) V^T with g(x) = x (3 - x^2) / 2, is the exact-arithmetic
 * result of k Newton-Schulz steps X <- 1/2 X (3I - X^2) from X0 = T/s; it is
 * obtained without any matrix product and is used to separate truncation error
 * (fixed iteration counts) from rounding error (reading A13).
 *
 * Parity pins (tests/test_oracle_pins.py): closed forms (diagonal, 2x2,
 * tridiagonal Toeplitz), sign^2 = I, commutation, LAPACK eigh, full-coverage
 * limit == full-matrix sign, Tr D == number of negative eigenvalues counted by
 * LDL^T inertia, block-diagonal limit, locality, brute-force pattern.
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_OK 0
#define ORC_BAD_ARG (-1)
#define ORC_BAD_PATTERN (-3)

/* ------------------------------------------------------------------ pattern */

static int find_in_row(const int32_t *row_ptr, const int32_t *col_idx, int32_t row, int32_t col)
{
    int32_t lo = row_ptr[row], hi = row_ptr[row + 1] - 1;
    while (lo <= hi) {
        int32_t mid = lo + (hi - lo) / 2;
        if (col_idx[mid] == col) return mid;
        if (col_idx[mid] < col) lo = mid + 1; else hi = mid - 1;
    }
    return -1;
}

/* Reading A5: columns strictly ascending per row, diagonal block present,
 * pattern structurally symmetric; else -3. */
int orc_check_pattern(int32_t n_blk, const int32_t *row_ptr, const int32_t *col_idx)
{
    if (n_blk < 0 || row_ptr[0] != 0) return ORC_BAD_ARG;
    for (int32_t i = 0; i < n_blk; ++i) {
        if (row_ptr[i + 1] < row_ptr[i]) return ORC_BAD_ARG;
        int has_diag = 0;
        for (int32_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int32_t j = col_idx[p];
            if (j < 0 || j >= n_blk) return ORC_BAD_ARG;
            if (p > row_ptr[i] && col_idx[p - 1] >= j) return ORC_BAD_PATTERN;
            if (j == i) has_diag = 1;
            if (find_in_row(row_ptr, col_idx, j, i) < 0) return ORC_BAD_PATTERN;
        }
        if (!has_diag) return ORC_BAD_PATTERN;
    }
    return ORC_OK;
}

static int32_t round_up(int32_t x, int32_t to) { return ((x + to - 1) / to) * to; }

/* N(i) = { j : block (j,i) is stored }, ascending (PAPER.md:110 step 1, reading A2):
 * walk the rows j in ascending order and append j to the list of every column it
 * stores.  out[0]=nbr_len out[1]=gmap_len out[2]=packed_elems out[3]=max_dim
 * out[4]=max_dim_pad */
int orc_pattern_sizes(int32_t n_blk, const int32_t *blk_size, const int32_t *row_ptr,
                      const int32_t *col_idx, int32_t pad_to, int64_t *out)
{
    if (pad_to <= 0) return ORC_BAD_ARG;
    int64_t *dim = (int64_t *)calloc((size_t)n_blk + 1, sizeof(int64_t));
    int64_t *cnt = (int64_t *)calloc((size_t)n_blk + 1, sizeof(int64_t));
    for (int32_t j = 0; j < n_blk; ++j)
        for (int32_t p = row_ptr[j]; p < row_ptr[j + 1]; ++p) {
            dim[col_idx[p]] += blk_size[j];
            cnt[col_idx[p]] += 1;
        }
    int64_t nbr = 0, gm = 0, pk = 0, md = 0, mdp = 0;
    for (int32_t i = 0; i < n_blk; ++i) {
        int64_t dp = round_up((int32_t)dim[i], pad_to);
        nbr += cnt[i]; gm += cnt[i] * cnt[i]; pk += dp * dp;
        if (dim[i] > md) md = dim[i];
        if (dp > mdp) mdp = dp;
    }
    out[0] = nbr; out[1] = gm; out[2] = pk; out[3] = md; out[4] = mdp;
    free(dim); free(cnt);
    return ORC_OK;
}

int orc_build_pattern(int32_t n_blk, const int32_t *blk_size, const int32_t *row_ptr,
                      const int32_t *col_idx, int32_t pad_to,
                      int32_t *nbr_ptr, int32_t *nbr_idx, int32_t *own_pos, int32_t *dim,
                      int32_t *dim_pad, int32_t *row_off, int64_t *sub_off, int64_t *gmap_ptr,
                      int32_t *gmap, int32_t *tmap, int32_t *order)
{
    if (pad_to <= 0) return ORC_BAD_ARG;
    int rc = orc_check_pattern(n_blk, row_ptr, col_idx);
    if (rc != ORC_OK) return rc;
    /* column lists */
    int32_t *fill = (int32_t *)calloc((size_t)n_blk + 1, sizeof(int32_t));
    for (int32_t i = 0; i <= n_blk; ++i) nbr_ptr[i] = 0;
    for (int32_t j = 0; j < n_blk; ++j)
        for (int32_t p = row_ptr[j]; p < row_ptr[j + 1]; ++p) nbr_ptr[col_idx[p] + 1] += 1;
    for (int32_t i = 0; i < n_blk; ++i) nbr_ptr[i + 1] += nbr_ptr[i];
    for (int32_t j = 0; j < n_blk; ++j)
        for (int32_t p = row_ptr[j]; p < row_ptr[j + 1]; ++p) {
            int32_t c = col_idx[p];
            nbr_idx[nbr_ptr[c] + fill[c]] = j;
            fill[c] += 1;
        }
    free(fill);
    sub_off[0] = 0; gmap_ptr[0] = 0;
    for (int32_t i = 0; i < n_blk; ++i) {
        int32_t cnt = nbr_ptr[i + 1] - nbr_ptr[i];
        int32_t off = 0; own_pos[i] = -1;
        for (int32_t a = 0; a < cnt; ++a) {
            int32_t j = nbr_idx[nbr_ptr[i] + a];
            if (j == i) own_pos[i] = a;
            row_off[nbr_ptr[i] + a] = off;
            off += blk_size[j];
        }
        dim[i] = off;
        dim_pad[i] = round_up(off, pad_to);
        sub_off[i + 1] = sub_off[i] + (int64_t)dim_pad[i] * dim_pad[i];
        gmap_ptr[i + 1] = gmap_ptr[i] + (int64_t)cnt * cnt;
        /* gather map: stored-block index of (N(i)[a], N(i)[c]) or -1 */
        for (int32_t a = 0; a < cnt; ++a)
            for (int32_t c = 0; c < cnt; ++c)
                gmap[gmap_ptr[i] + (int64_t)a * cnt + c] =
                    find_in_row(row_ptr, col_idx, nbr_idx[nbr_ptr[i] + a], nbr_idx[nbr_ptr[i] + c]);
    }
    /* transpose map: index of block (j,i) for p = (i,j) */
    for (int32_t i = 0; i < n_blk; ++i)
        for (int32_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p)
            tmap[p] = find_in_row(row_ptr, col_idx, col_idx[p], i);
    /* schedule: (dim_pad descending, id ascending) -- stable insertion of ids */
    for (int32_t i = 0; i < n_blk; ++i) order[i] = i;
    /* simple stable merge sort on key -dim_pad */
    int32_t *tmp = (int32_t *)malloc((size_t)(n_blk > 0 ? n_blk : 1) * sizeof(int32_t));
    for (int32_t w = 1; w < n_blk; w *= 2) {
        for (int32_t lo = 0; lo < n_blk; lo += 2 * w) {
            int32_t mid = lo + w < n_blk ? lo + w : n_blk;
            int32_t hi = lo + 2 * w < n_blk ? lo + 2 * w : n_blk;
            int32_t a = lo, b = mid, k = lo;
            while (a < mid && b < hi)
                tmp[k++] = (dim_pad[order[b]] > dim_pad[order[a]]) ? order[b++] : order[a++];
            while (a < mid) tmp[k++] = order[a++];
            while (b < hi) tmp[k++] = order[b++];
        }
        memcpy(order, tmp, (size_t)n_blk * sizeof(int32_t));
    }
    free(tmp);
    return ORC_OK;
}

/* --------------------------------------------------------------- step 1: gather */

/* T (m x m, row-major) = principal submatrix of A on N(i), minus mu*I.
 * Absent block pairs are zero (reading A2); PAPER.md:91 for the shift. */
int orc_gather(int32_t n_blk, const int32_t *blk_size, const int32_t *row_ptr,
               const int32_t *col_idx, const int64_t *val_ptr, const double *vals,
               int32_t i, double mu, double *T)
{
    (void)n_blk;
    /* N(i): by structural symmetry (checked by the caller) the rows storing column i
     * are the columns stored in row i. */
    int32_t cnt = row_ptr[i + 1] - row_ptr[i];
    const int32_t *nb = col_idx + row_ptr[i];
    int32_t m = 0;
    for (int32_t a = 0; a < cnt; ++a) m += blk_size[nb[a]];
    memset(T, 0, (size_t)m * m * sizeof(double));
    int32_t ro = 0;
    for (int32_t a = 0; a < cnt; ++a) {
        int32_t ja = nb[a], ba = blk_size[ja], co = 0;
        for (int32_t c = 0; c < cnt; ++c) {
            int32_t jc = nb[c], bc = blk_size[jc];
            int32_t p = find_in_row(row_ptr, col_idx, ja, jc);
            if (p >= 0) {
                const double *blk = vals + val_ptr[p];
                for (int32_t r = 0; r < ba; ++r)
                    for (int32_t s = 0; s < bc; ++s)
                        T[(size_t)(ro + r) * m + (co + s)] = blk[(size_t)r * bc + s];
            }
            co += bc;
        }
        ro += ba;
    }
    for (int32_t r = 0; r < m; ++r) T[(size_t)r * m + r] -= mu;
    return m;
}

/* Gershgorin bound on the spectral radius: max_r sum_c |T_rc| (reading A10). */
double orc_gershgorin(int32_t m, const double *T)
{
    double s = 0.0;
    for (int32_t r = 0; r < m; ++r) {
        double row = 0.0;
        for (int32_t c = 0; c < m; ++c) row += fabs(T[(size_t)r * m + c]);
        if (row > s) s = row;
    }
    return s;
}

/* -------------------------------------------------- step 2: f = sign via Jacobi */

/* Cyclic Jacobi eigendecomposition of symmetric A (m x m, row-major, destroyed).
 * On return w[k] = eigenvalues, Vt row k = eigenvector k (A = Vt^T diag(w) Vt).
 * Stops when off(A)^2 <= rel_tol^2 ||A||_F^2 or after max_sweeps.  Returns sweeps. */
int orc_jacobi(int32_t m, double *A, double *Vt, double *w, int32_t max_sweeps, double rel_tol)
{
    for (int32_t r = 0; r < m; ++r)
        for (int32_t c = 0; c < m; ++c) Vt[(size_t)r * m + c] = (r == c) ? 1.0 : 0.0;
    double fro2 = 0.0;
    for (size_t k = 0; k < (size_t)m * m; ++k) fro2 += A[k] * A[k];
    int sweep = 0;
    for (; sweep < max_sweeps; ++sweep) {
        double off2 = 0.0;
        for (int32_t p = 0; p < m; ++p)
            for (int32_t q = p + 1; q < m; ++q) off2 += 2.0 * A[(size_t)p * m + q] * A[(size_t)p * m + q];
        if (off2 <= rel_tol * rel_tol * fro2) break;
        for (int32_t p = 0; p < m - 1; ++p) {
            for (int32_t q = p + 1; q < m; ++q) {
                double apq = A[(size_t)p * m + q];
                if (apq == 0.0) continue;
                double app = A[(size_t)p * m + p], aqq = A[(size_t)q * m + q];
                double theta = (aqq - app) / (2.0 * apq);
                double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
                double *Ap = A + (size_t)p * m, *Aq = A + (size_t)q * m;
                /* rows p and q of J^T A J (k != p,q), J = rotation in the (p,q) plane */
                for (int32_t k = 0; k < m; ++k) {
                    double x = Ap[k], y = Aq[k];
                    Ap[k] = c * x - s * y;
                    Aq[k] = s * x + c * y;
                }
                /* the 2x2 pivot block in closed form; a_pq is annihilated */
                Ap[p] = app - t * apq;
                Aq[q] = aqq + t * apq;
                Ap[q] = 0.0;
                Aq[p] = 0.0;
                /* columns p and q follow by symmetry */
                for (int32_t k = 0; k < m; ++k) {
                    if (k == p || k == q) continue;
                    A[(size_t)k * m + p] = Ap[k];
                    A[(size_t)k * m + q] = Aq[k];
                }
                double *Vp = Vt + (size_t)p * m, *Vq = Vt + (size_t)q * m;
                for (int32_t k = 0; k < m; ++k) {
                    double x = Vp[k], y = Vq[k];
                    Vp[k] = c * x - s * y;
                    Vq[k] = s * x + c * y;
                }
            }
        }
    }
    for (int32_t k = 0; k < m; ++k) w[k] = A[(size_t)k * m + k];
    return sweep;
}

/* S = sum_k f_k v_k v_k^T, v_k = row k of Vt. */
static void spectral_sum(int32_t m, const double *Vt, const double *f, double *S)
{
    memset(S, 0, (size_t)m * m * sizeof(double));
    for (int32_t k = 0; k < m; ++k) {
        const double *v = Vt + (size_t)k * m;
        double fk = f[k];
        if (fk == 0.0) continue;
        for (int32_t r = 0; r < m; ++r) {
            double a = fk * v[r];
            double *Sr = S + (size_t)r * m;
            for (int32_t c = 0; c < m; ++c) Sr[c] += a * v[c];
        }
    }
}

/* Eq. 13 by its definition on the spectrum: sign(T) = V diag(sgn w) V^T, sgn(0) := 0. */
void orc_sign_from_eig(int32_t m, const double *Vt, const double *w, double *S)
{
    double *f = (double *)malloc((size_t)(m > 0 ? m : 1) * sizeof(double));
    for (int32_t k = 0; k < m; ++k) f[k] = (w[k] > 0.0) ? 1.0 : ((w[k] < 0.0) ? -1.0 : 0.0);
    spectral_sum(m, Vt, f, S);
    free(f);
}

/* NS-k polynomial: V diag(g^k(w/scale)) V^T, g(x) = x(3 - x^2)/2 (reading A9/A13). */
void orc_nsk_from_eig(int32_t m, const double *Vt, const double *w, double scale, int32_t k,
                      double *S)
{
    double *f = (double *)malloc((size_t)(m > 0 ? m : 1) * sizeof(double));
    for (int32_t e = 0; e < m; ++e) {
        double x = w[e] / scale;
        for (int32_t it = 0; it < k; ++it) x = 0.5 * x * (3.0 - x * x);
        f[e] = x;
    }
    spectral_sum(m, Vt, f, S);
    free(f);
}

/* Third-order iteration, k steps ("various iterative methods", reading A22 in
 * DESIGN.md): V diag(g3^k(w/scale)) V^T with g3(x) = x (15 - 10 x^2 + 3 x^4) / 8, the next member after
 * g(x) = x (3 - x^2) / 2 of the family x (1 - w)^-1/2, w = 1 - x^2, truncated after w^2:
 * x (1 + w/2 + 3 w^2 / 8).  Fixed points 0, +-1, +-sqrt(7/3); g3' = g3'' = 0 at +-1 (cubic convergence);
 * converges to sgn(x) for 0 < |x| < sqrt(7/3). */
void orc_ns3k_from_eig(int32_t m, const double *Vt, const double *w, double scale, int32_t k,
                       double *S)
{
    double *f = (double *)malloc((size_t)(m > 0 ? m : 1) * sizeof(double));
    for (int32_t e = 0; e < m; ++e) {
        double x = w[e] / scale;
        for (int32_t it = 0; it < k; ++it) {
            double x2 = x * x;
            x = x * (15.0 - 10.0 * x2 + 3.0 * x2 * x2) / 8.0;
        }
        f[e] = x;
    }
    spectral_sum(m, Vt, f, S);
    free(f);
}

/* --------------------------- steps 1-3 + Eq. 14 for a list of block columns */

typedef struct {
    int32_t n_blk;
    const int32_t *blk_size, *row_ptr, *col_idx;
    const int64_t *val_ptr;
    const double *vals;
    double mu;
    int32_t n_cols;
    const int32_t *cols;
    int32_t mode;          /* 0: exact sign; 1: NS-k polynomial with Gershgorin scale; 2: third-order, k steps */
    int32_t k_fixed;
    const double *scale_in; /* mode 1: optional per-column scale (NULL -> Gershgorin) */
    double *d_vals;        /* out: D = 1/2 (I - S) blocks of the listed columns, A's layout */
    double *min_abs_eig;   /* out [n_cols] */
    double *scale_out;     /* out [n_cols] Gershgorin bound of T_i - mu I */
    int32_t *sweeps;       /* out [n_cols] */
    int32_t *n_neg;        /* out [n_cols] number of negative eigenvalues of T_i - mu I */
    int32_t next;          /* work counter */
    pthread_mutex_t lock;
} orc_job_t;

static void density_one(orc_job_t *J, int32_t ci)
{
    int32_t i = J->cols ? J->cols[ci] : ci;
    int32_t cnt = J->row_ptr[i + 1] - J->row_ptr[i];
    const int32_t *nb = J->col_idx + J->row_ptr[i];
    int32_t m = 0;
    for (int32_t a = 0; a < cnt; ++a) m += J->blk_size[nb[a]];
    size_t mm = (size_t)m * m;
    double *T = (double *)malloc(mm * sizeof(double));
    double *Vt = (double *)malloc(mm * sizeof(double));
    double *S = (double *)malloc(mm * sizeof(double));
    double *w = (double *)malloc((size_t)m * sizeof(double));
    orc_gather(J->n_blk, J->blk_size, J->row_ptr, J->col_idx, J->val_ptr, J->vals, i, J->mu, T);
    double gs = orc_gershgorin(m, T);
    int sw = orc_jacobi(m, T, Vt, w, 30, 1e-15);
    double mn = INFINITY; int32_t nneg = 0;
    for (int32_t k = 0; k < m; ++k) { if (fabs(w[k]) < mn) mn = fabs(w[k]); if (w[k] < 0.0) ++nneg; }
    if (J->mode == 0) orc_sign_from_eig(m, Vt, w, S);
    else if (J->mode == 2) orc_ns3k_from_eig(m, Vt, w, J->scale_in ? J->scale_in[ci] : gs, J->k_fixed, S);
    else orc_nsk_from_eig(m, Vt, w, J->scale_in ? J->scale_in[ci] : gs, J->k_fixed, S);
    /* step 3: rows = all of N(i), columns = local position of block i.
     * By structural symmetry block (N(i)[a'], i) is found in row N(i)[a']. */
    int32_t own = -1, own_off = 0, ro = 0;
    for (int32_t a = 0; a < cnt; ++a) { if (nb[a] == i) { own = a; own_off = ro; } ro += J->blk_size[nb[a]]; }
    int32_t bi = J->blk_size[i];
    ro = 0;
    for (int32_t a = 0; a < cnt; ++a) {
        int32_t j = nb[a], bj = J->blk_size[j];
        int32_t p = find_in_row(J->row_ptr, J->col_idx, j, i);
        double *blk = J->d_vals + J->val_ptr[p];
        for (int32_t r = 0; r < bj; ++r)
            for (int32_t s = 0; s < bi; ++s) {
                double sv = S[(size_t)(ro + r) * m + (own_off + s)];
                double id = (a == own && r == s) ? 1.0 : 0.0;
                blk[(size_t)r * bi + s] = 0.5 * (id - sv);   /* Eq. 14, S = I */
            }
        ro += bj;
    }
    if (J->min_abs_eig) J->min_abs_eig[ci] = mn;
    if (J->scale_out) J->scale_out[ci] = gs;
    if (J->sweeps) J->sweeps[ci] = sw;
    if (J->n_neg) J->n_neg[ci] = nneg;
    free(T); free(Vt); free(S); free(w);
}

static void *density_worker(void *arg)
{
    orc_job_t *J = (orc_job_t *)arg;
    for (;;) {
        pthread_mutex_lock(&J->lock);
        int32_t ci = J->next++;
        pthread_mutex_unlock(&J->lock);
        if (ci >= J->n_cols) break;
        density_one(J, ci);
    }
    return NULL;
}

/* Raw (unsymmetrised) density blocks of the listed block columns; blocks of other
 * columns in d_vals are left untouched.  cols == NULL: all columns. */
int orc_density_columns(int32_t n_blk, const int32_t *blk_size, const int32_t *row_ptr,
                        const int32_t *col_idx, const int64_t *val_ptr, const double *vals,
                        double mu, int32_t n_cols, const int32_t *cols, int32_t mode,
                        int32_t k_fixed, const double *scale_in, double *d_vals,
                        double *min_abs_eig, double *scale_out, int32_t *sweeps, int32_t *n_neg,
                        int32_t n_threads)
{
    int rc = orc_check_pattern(n_blk, row_ptr, col_idx);
    if (rc != ORC_OK) return rc;
    orc_job_t J;
    J.n_blk = n_blk; J.blk_size = blk_size; J.row_ptr = row_ptr; J.col_idx = col_idx;
    J.val_ptr = val_ptr; J.vals = vals; J.mu = mu; J.n_cols = cols ? n_cols : n_blk; J.cols = cols;
    J.mode = mode; J.k_fixed = k_fixed; J.scale_in = scale_in; J.d_vals = d_vals;
    J.min_abs_eig = min_abs_eig; J.scale_out = scale_out; J.sweeps = sweeps; J.n_neg = n_neg;
    J.next = 0;
    pthread_mutex_init(&J.lock, NULL);
    if (n_threads < 1) n_threads = 1;
    if (n_threads > 256) n_threads = 256;
    pthread_t th[256];
    for (int t = 1; t < n_threads; ++t) pthread_create(&th[t], NULL, density_worker, &J);
    density_worker(&J);
    for (int t = 1; t < n_threads; ++t) pthread_join(th[t], NULL);
    pthread_mutex_destroy(&J.lock);
    return ORC_OK;
}

/* D_sym = 1/2 (D + D^T) blockwise through the transpose map (reading A6). */
int orc_symmetrise(int32_t n_blk, const int32_t *blk_size, const int32_t *row_ptr,
                   const int32_t *col_idx, const int64_t *val_ptr, const double *d_raw,
                   double *d_sym)
{
    for (int32_t i = 0; i < n_blk; ++i)
        for (int32_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            int32_t j = col_idx[p];
            int32_t q = find_in_row(row_ptr, col_idx, j, i);
            if (q < 0) return ORC_BAD_PATTERN;
            int32_t bi = blk_size[i], bj = blk_size[j];
            const double *a = d_raw + val_ptr[p], *b = d_raw + val_ptr[q];
            double *o = d_sym + val_ptr[p];
            for (int32_t r = 0; r < bi; ++r)
                for (int32_t s = 0; s < bj; ++s)
                    o[(size_t)r * bj + s] = 0.5 * (a[(size_t)r * bj + s] + b[(size_t)s * bi + r]);
        }
    return ORC_OK;
}

/* Tr D = sum of the diagonals of the diagonal blocks. */
double orc_trace(int32_t n_blk, const int32_t *blk_size, const int32_t *row_ptr,
                 const int32_t *col_idx, const int64_t *val_ptr, const double *d_vals)
{
    double tr = 0.0;
    for (int32_t i = 0; i < n_blk; ++i) {
        int32_t p = find_in_row(row_ptr, col_idx, i, i);
        if (p < 0) continue;
        int32_t b = blk_size[i];
        for (int32_t r = 0; r < b; ++r) tr += d_vals[val_ptr[p] + (size_t)r * b + r];
    }
    return tr;
}
