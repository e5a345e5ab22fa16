/*
 * sharp_oracle.c -- CPU ORACLE for the ptychographic projection loop of arXiv 1602.01448 (SHARP).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference leg may build, load or call it.  It shares no code, header, table or
 * helper with the CUDA path under paper_1602_01448_b200/csrc/ and neither includes the other.
 *
 * Plain C99, double precision, one loop nest per formula, in the paper's order and notation:
 *   psi  object  (n_r x n_c complex)
 *   w    illumination (m x m complex)
 *   z    frames  (K x m x m complex)        PAPER.md:66-68, Eq. (5) at :127
 *   a    amplitudes sqrt(I) (K x m x m)
 *   x_i  integer translations (row, col) of the frame's top-left pixel, in {0..n-m}
 * No blocking, fusion or reordering beyond what the definitions state.  "#pragma omp parallel for" is put
 * only on loops whose iterations are independent (over frames, or over object rows); every sum is taken
 * serially in the stated order (ascending frame index i for sums over frames, reading G17).
 *
 * Readings of the paper used here (DESIGN.md section "Readings"): G1 RAAR sign, G2 DFT sign, G3 unitary
 * scaling, G4 small-|Fz| rule, G5 uncovered pixels, G7 z0, G10 step order when refining w.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): DFT vs closed forms / Parseval / an independent library
 * FFT; Q,Q* adjointness; P_Q vs a dense matrix built from Eq. (5); projector idempotence; RAAR fixed point,
 * beta=1 Douglas-Rachford, literal vs one-overlap form; probe update closed forms; metric invariances;
 * tile lists vs interval arithmetic.  Parity unpinned: the absolute trajectory of the chaotic configs
 * beyond ~10 iterations.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

static const double ORC_PI = 3.14159265358979323846264338327950288;

/* ------------------------------------------------------------------------------------------------
 * O1  the 2-D DFT, Eq. (2) PAPER.md:62-64 with reading G2 (forward kernel e^{-2 pi i q.r}) and the
 *     unitary scale 1/sqrt(m^2) = 1/m per 2-D transform (G3).  sign = -1 forward F, +1 adjoint F*.
 *
 *   (F f)(u,v) = (1/m) sum_{r,c} f(r,c) exp(sign * 2 pi i (u r + v c)/m),   u,v,r,c in {0..m-1}
 *
 * orc_dft2_naive is this definition evaluated as two nested 1-D sums (rows, then columns); the twiddle
 * angle uses the reduced integer (u*r mod m) so that it is exact for every index.
 * ---------------------------------------------------------------------------------------------- */
static void dft1_naive(int m, const cplx *in, int istride, cplx *out, int ostride, int sign)
{
    for (int u = 0; u < m; ++u) {
        cplx acc = 0.0;
        for (int r = 0; r < m; ++r) {
            int k = (int)(((long)u * r) % m);
            double ang = sign * 2.0 * ORC_PI * (double)k / (double)m;
            acc += in[(long)r * istride] * (cos(ang) + I * sin(ang));
        }
        out[(long)u * ostride] = acc;
    }
}

void orc_dft2_naive(int m, const cplx *in, cplx *out, int sign)
{
    cplx *tmp = (cplx *)malloc(sizeof(cplx) * (size_t)m * m);
    /* transform along c (each row), then along r (each column) */
    for (int r = 0; r < m; ++r) dft1_naive(m, in + (long)r * m, 1, tmp + (long)r * m, 1, sign);
    for (int c = 0; c < m; ++c) dft1_naive(m, tmp + c, m, out + c, m, sign);
    for (long j = 0; j < (long)m * m; ++j) out[j] /= (double)m;
    free(tmp);
}

/* Own radix-2 decimation-in-time FFT (textbook Cooley-Tukey: bit-reversal permutation, then log2 m
 * butterfly stages).  Used for speed; orc_dft2_naive checks it (tests/test_oracle_dft.py).  m must be a
 * power of two. */
static void fft1_radix2(int m, cplx *x, int sign)
{
    for (int i = 1, j = 0; i < m; ++i) {          /* bit reversal */
        int bit = m >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = x[i]; x[i] = x[j]; x[j] = t; }
    }
    for (int len = 2; len <= m; len <<= 1) {
        int half = len >> 1;
        for (int s = 0; s < m; s += len) {
            for (int k = 0; k < half; ++k) {
                double ang = sign * 2.0 * ORC_PI * (double)k / (double)len;
                cplx tw = cos(ang) + I * sin(ang);
                cplx e = x[s + k], o = x[s + k + half] * tw;
                x[s + k] = e + o;
                x[s + k + half] = e - o;
            }
        }
    }
}

void orc_fft2(int m, const cplx *in, cplx *out, int sign)
{
    cplx *col = (cplx *)malloc(sizeof(cplx) * (size_t)m);
    if (out != in) memcpy(out, in, sizeof(cplx) * (size_t)m * m);
    for (int r = 0; r < m; ++r) fft1_radix2(m, out + (long)r * m, sign);
    for (int c = 0; c < m; ++c) {
        for (int r = 0; r < m; ++r) col[r] = out[(long)r * m + c];
        fft1_radix2(m, col, sign);
        for (int r = 0; r < m; ++r) out[(long)r * m + c] = col[r] / (double)m;
    }
    free(col);
}

/* ------------------------------------------------------------------------------------------------
 * O2  amplitudes a = sqrt(I), negatives clamped (G14); A2 = sum a^2 = ||a||^2 (G12).
 * ---------------------------------------------------------------------------------------------- */
void orc_amplitudes(long n, const float *Iq, double *a, double *A2)
{
    double s = 0.0;
    for (long j = 0; j < n; ++j) {
        double v = (double)Iq[j];
        if (v < 0.0) v = 0.0;
        a[j] = sqrt(v);
        s += v;
    }
    *A2 = s;
}

/* ------------------------------------------------------------------------------------------------
 * O3  split: z_i(r) = w(r) psi(r + x_i)            PAPER.md:66-68 (Q_i = diag(w) T_i)
 * ---------------------------------------------------------------------------------------------- */
void orc_split(int m, int K, const int32_t *pos, int nr, int nc, const cplx *psi, const cplx *w, cplx *z)
{
    (void)nr;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < K; ++i)
        for (int r = 0; r < m; ++r)
            for (int c = 0; c < m; ++c)
                z[((long)i * m + r) * m + c] =
                    w[(long)r * m + c] * psi[(long)(pos[2 * i] + r) * nc + (pos[2 * i + 1] + c)];
}

/* ------------------------------------------------------------------------------------------------
 * O4  overlap: (Q* f)(p) = sum_i conj(w(p - x_i)) f_i(p - x_i)      PAPER.md:153-155 (numerator of Eq. 9)
 *              (Q* Q)(p) = sum_i |w(p - x_i)|^2                      (denominator of Eq. 9)
 *     The sum over frames runs in ascending i (G17).  Written scatter-wise, frame after frame, which for a
 *     serial loop gives every pixel its contributions in ascending i.
 * ---------------------------------------------------------------------------------------------- */
void orc_overlap_num(int m, int K, const int32_t *pos, int nr, int nc, const cplx *w, const cplx *f, cplx *num)
{
    for (long p = 0; p < (long)nr * nc; ++p) num[p] = 0.0;
    for (int i = 0; i < K; ++i)
        for (int r = 0; r < m; ++r)
            for (int c = 0; c < m; ++c)
                num[(long)(pos[2 * i] + r) * nc + (pos[2 * i + 1] + c)] +=
                    conj(w[(long)r * m + c]) * f[((long)i * m + r) * m + c];
}

void orc_overlap_den(int m, int K, const int32_t *pos, int nr, int nc, const cplx *w, double *den)
{
    for (long p = 0; p < (long)nr * nc; ++p) den[p] = 0.0;
    for (int i = 0; i < K; ++i)
        for (int r = 0; r < m; ++r)
            for (int c = 0; c < m; ++c) {
                cplx wv = w[(long)r * m + c];
                den[(long)(pos[2 * i] + r) * nc + (pos[2 * i + 1] + c)] +=
                    creal(wv) * creal(wv) + cimag(wv) * cimag(wv);
            }
}

/* L_w f = (Q*Q)^{-1} Q* f, Eq. (9); psi(p) = 0 where Q*Q(p) = 0 (G5). */
void orc_L(int m, int K, const int32_t *pos, int nr, int nc, const cplx *w, const cplx *f, cplx *psi)
{
    double *den = (double *)malloc(sizeof(double) * (size_t)nr * nc);
    orc_overlap_num(m, K, pos, nr, nc, w, f, psi);
    orc_overlap_den(m, K, pos, nr, nc, w, den);
    for (long p = 0; p < (long)nr * nc; ++p) psi[p] = (den[p] > 0.0) ? psi[p] / den[p] : 0.0;
    free(den);
}

/* P_Q f = Q (Q*Q)^{-1} Q* f, Eq. (8) */
void orc_PQ(int m, int K, const int32_t *pos, int nr, int nc, const cplx *w, const cplx *f, cplx *out)
{
    cplx *psi = (cplx *)malloc(sizeof(cplx) * (size_t)nr * nc);
    orc_L(m, K, pos, nr, nc, w, f, psi);
    orc_split(m, K, pos, nr, nc, psi, w, out);
    free(psi);
}

/* ------------------------------------------------------------------------------------------------
 * O5  data projector, Eq. (7):  P_a z = F* [ (F z / |F z|) a ]
 *     G4: where |F z| <= thr the phase factor is taken as 1 (Z' = a).
 *     use_naive != 0 selects the O(m^3) DFT instead of the radix-2 one (small cases only).
 * ---------------------------------------------------------------------------------------------- */
void orc_Pa(int m, int K, const cplx *z, const double *a, double thr, cplx *y, int use_naive)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < K; ++i) {
        long off = (long)i * m * m;
        cplx *Z = (cplx *)malloc(sizeof(cplx) * (size_t)m * m);
        if (use_naive) orc_dft2_naive(m, z + off, Z, -1); else orc_fft2(m, z + off, Z, -1);
        for (long q = 0; q < (long)m * m; ++q) {
            double mag = cabs(Z[q]);
            Z[q] = (mag > thr) ? (Z[q] / mag) * a[off + q] : (cplx)a[off + q];
        }
        if (use_naive) orc_dft2_naive(m, Z, y + off, +1); else orc_fft2(m, Z, y + off, +1);
        free(Z);
    }
}

/* ------------------------------------------------------------------------------------------------
 * O6  RAAR, step 5 PAPER.md:174-178 with the sign of reading G1 (Luke [60]):
 *        z' = [ 2 beta P_Q P_a + (1 - 2 beta) P_a + beta (I - P_Q) ] z
 *     Evaluated literally: y = P_a z, then the two overlap projections P_Q y and P_Q z.
 *     y_out (may be NULL) receives P_a z.
 * ---------------------------------------------------------------------------------------------- */
void orc_raar(int m, int K, const int32_t *pos, int nr, int nc, const cplx *w, const double *a, double thr,
              double beta, const cplx *z, cplx *znew, cplx *y_out, int use_naive)
{
    long N = (long)K * m * m;
    cplx *y = (cplx *)malloc(sizeof(cplx) * (size_t)N);
    cplx *PQy = (cplx *)malloc(sizeof(cplx) * (size_t)N);
    cplx *PQz = (cplx *)malloc(sizeof(cplx) * (size_t)N);
    orc_Pa(m, K, z, a, thr, y, use_naive);
    orc_PQ(m, K, pos, nr, nc, w, y, PQy);
    orc_PQ(m, K, pos, nr, nc, w, z, PQz);
    for (long j = 0; j < N; ++j)
        znew[j] = 2.0 * beta * PQy[j] + (1.0 - 2.0 * beta) * y[j] + beta * (z[j] - PQz[j]);
    if (y_out) memcpy(y_out, y, sizeof(cplx) * (size_t)N);
    free(y); free(PQy); free(PQz);
}

/* The same step written with one split:  z' = beta Q(2 L y - L z) + (1 - 2 beta) y + beta z.
 * Present only so that a test can assert it equals orc_raar. */
void orc_raar_one_split(int m, int K, const int32_t *pos, int nr, int nc, const cplx *w, const double *a,
                        double thr, double beta, const cplx *z, cplx *znew, int use_naive)
{
    long N = (long)K * m * m, P = (long)nr * nc;
    cplx *y = (cplx *)malloc(sizeof(cplx) * (size_t)N);
    cplx *q = (cplx *)malloc(sizeof(cplx) * (size_t)N);
    cplx *py = (cplx *)malloc(sizeof(cplx) * (size_t)P);
    cplx *pz = (cplx *)malloc(sizeof(cplx) * (size_t)P);
    orc_Pa(m, K, z, a, thr, y, use_naive);
    orc_L(m, K, pos, nr, nc, w, y, py);
    orc_L(m, K, pos, nr, nc, w, z, pz);
    for (long p = 0; p < P; ++p) py[p] = 2.0 * py[p] - pz[p];
    orc_split(m, K, pos, nr, nc, py, w, q);
    for (long j = 0; j < N; ++j) znew[j] = beta * q[j] + (1.0 - 2.0 * beta) * y[j] + beta * z[j];
    free(y); free(q); free(py); free(pz);
}

/* ------------------------------------------------------------------------------------------------
 * O8  illumination update, Eq. (10) PAPER.md:157-159:
 *        w(r) <- sum_i conj(psi(r + x_i)) z_i(r) / sum_i |psi(r + x_i)|^2      (ascending i)
 *     where the denominator is 0 the old w(r) is kept.
 * ---------------------------------------------------------------------------------------------- */
void orc_probe_update(int m, int K, const int32_t *pos, int nr, int nc, const cplx *psi, const cplx *z, cplx *w)
{
    (void)nr;
#pragma omp parallel for schedule(static)
    for (int r = 0; r < m; ++r)
        for (int c = 0; c < m; ++c) {
            cplx num = 0.0;
            double den = 0.0;
            for (int i = 0; i < K; ++i) {
                cplx pv = psi[(long)(pos[2 * i] + r) * nc + (pos[2 * i + 1] + c)];
                num += conj(pv) * z[((long)i * m + r) * m + c];
                den += creal(pv) * creal(pv) + cimag(pv) * cimag(pv);
            }
            if (den > 0.0) w[(long)r * m + c] = num / den;
        }
}

/* ------------------------------------------------------------------------------------------------
 * O9  metrics, Eq. (11)-(13) PAPER.md:196-206 (G12: plain ratios of 2-norms, ||a|| = sqrt(A2)):
 *        eps_a = ||P_a z - z|| / ||a||,  eps_Q = ||P_Q z - z|| / ||a||,  eps_D = ||z - zprev|| / ||a||
 *     zprev == NULL means z^(l-1) = 0 (reading G7).
 * ---------------------------------------------------------------------------------------------- */
void orc_errors(int m, int K, const int32_t *pos, int nr, int nc, const cplx *w, const double *a, double thr,
                double A2, const cplx *z, const cplx *zprev, double out[3], int use_naive)
{
    long N = (long)K * m * m;
    cplx *t = (cplx *)malloc(sizeof(cplx) * (size_t)N);
    double sa = 0.0, sq = 0.0, sd = 0.0;
    orc_Pa(m, K, z, a, thr, t, use_naive);
    for (long j = 0; j < N; ++j) { cplx d = t[j] - z[j]; sa += creal(d) * creal(d) + cimag(d) * cimag(d); }
    orc_PQ(m, K, pos, nr, nc, w, z, t);
    for (long j = 0; j < N; ++j) { cplx d = t[j] - z[j]; sq += creal(d) * creal(d) + cimag(d) * cimag(d); }
    for (long j = 0; j < N; ++j) {
        cplx d = z[j] - (zprev ? zprev[j] : 0.0);
        sd += creal(d) * creal(d) + cimag(d) * cimag(d);
    }
    free(t);
    out[0] = sqrt(sa / A2); out[1] = sqrt(sq / A2); out[2] = sqrt(sd / A2);
}

/* ------------------------------------------------------------------------------------------------
 * O10 integer artefacts of the geometry (compared bit-exactly with the GPU library's plan):
 *   (i)   linear object index of frame pixel (i, r, c):  (x_i.row + r) * n_c + (x_i.col + c)
 *   (ii)  per-pixel cover count  #{ i : p in frame i }
 *   (iii) per-tile frame lists by brute force over every (tile, frame) pair: frame i is in tile (ty,tx) iff
 *         [x_i.row, x_i.row+m) meets [ty*T, (ty+1)*T) and likewise for columns; tiles row-major, frames
 *         ascending.  Call with frames == NULL to get the counts (tile_ptr), then again to fill.
 * ---------------------------------------------------------------------------------------------- */
void orc_linear_index(int m, int K, const int32_t *pos, int nc, int64_t *idx)
{
    for (int i = 0; i < K; ++i)
        for (int r = 0; r < m; ++r)
            for (int c = 0; c < m; ++c)
                idx[((long)i * m + r) * m + c] = (int64_t)(pos[2 * i] + r) * nc + (pos[2 * i + 1] + c);
}

void orc_cover_counts(int m, int K, const int32_t *pos, int nr, int nc, int32_t *count)
{
    for (long p = 0; p < (long)nr * nc; ++p) count[p] = 0;
    for (int i = 0; i < K; ++i)
        for (int r = 0; r < m; ++r)
            for (int c = 0; c < m; ++c)
                count[(long)(pos[2 * i] + r) * nc + (pos[2 * i + 1] + c)] += 1;
}

void orc_tile_lists(int m, int K, const int32_t *pos, int nr, int nc, int T, int32_t *tile_ptr, int32_t *frames)
{
    int ty_n = (nr + T - 1) / T, tx_n = (nc + T - 1) / T;
    int32_t n = 0;
    for (int ty = 0; ty < ty_n; ++ty)
        for (int tx = 0; tx < tx_n; ++tx) {
            tile_ptr[ty * tx_n + tx] = n;
            for (int i = 0; i < K; ++i) {
                int r0 = pos[2 * i], c0 = pos[2 * i + 1];
                int hit_r = (r0 < (ty + 1) * T) && (r0 + m > ty * T);
                int hit_c = (c0 < (tx + 1) * T) && (c0 + m > tx * T);
                if (hit_r && hit_c) { if (frames) frames[n] = i; ++n; }
            }
        }
    tile_ptr[ty_n * tx_n] = n;
}
