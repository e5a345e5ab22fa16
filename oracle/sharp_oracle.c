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
 * scaling, G4 small-|Fz| rule, G5 uncovered pixels, G7 z0, G10 step order when refining w, G21 default w0 at
 * the frame centre, G22-G23 centre of mass of |w|^2 / integer cyclic shift of w alone, G24 small-|Fw| rule,
 * G25 periodic T_i.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): DFT vs closed forms / Parseval / an independent library
 * FFT; Q,Q* adjointness; P_Q vs a dense matrix built from Eq. (5); projector idempotence; RAAR fixed point,
 * beta=1 Douglas-Rachford, literal vs one-overlap form; probe update closed forms; metric invariances;
 * tile lists vs interval arithmetic; eps_0 vs a brute-force scan over phi and the expanded closed form; default
 * probe returns a zero-phase pupil probe exactly; mask projection idempotent, |F w'| = a_w; re-centring moves a
 * displaced probe back by the known integer; periodic T_i vs numpy.roll.  Parity unpinned: the absolute trajectory of the chaotic configs
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
 * T_i: object pixel under frame pixel (r, c) of frame i.  PAPER.md:53 puts x_i in {0..n-m}, so r + x_i never
 * leaves the image.  The simulation of PAPER.md:248 (Fig. 3) uses "periodic boundary conditions to avoid edge
 * effects": x_i anywhere in {0..n-1} and r + x_i taken modulo the image size (reading G25).  The
 * modulo below is the identity for positions in {0..n-m}, so both cases are this one expression.
 * ---------------------------------------------------------------------------------------------- */
static long obj_index(const int32_t *pos, int i, int r, int c, int nr, int nc)
{
    return (long)((pos[2 * i] + r) % nr) * nc + ((pos[2 * i + 1] + c) % nc);
}

/* ------------------------------------------------------------------------------------------------
 * O3  split: z_i(r) = w(r) psi(r + x_i)            PAPER.md:66-68 (Q_i = diag(w) T_i)
 * ---------------------------------------------------------------------------------------------- */
void orc_split(int m, int K, const int32_t *pos, int nr, int nc, const cplx *psi, const cplx *w, cplx *z)
{
#pragma omp parallel for schedule(static)
    for (int i = 0; i < K; ++i)
        for (int r = 0; r < m; ++r)
            for (int c = 0; c < m; ++c)
                z[((long)i * m + r) * m + c] = w[(long)r * m + c] * psi[obj_index(pos, i, r, c, nr, nc)];
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
                num[obj_index(pos, i, r, c, nr, nc)] += conj(w[(long)r * m + c]) * f[((long)i * m + r) * m + c];
}

void orc_overlap_den(int m, int K, const int32_t *pos, int nr, int nc, const cplx *w, double *den)
{
    for (long p = 0; p < (long)nr * nc; ++p) den[p] = 0.0;
    for (int i = 0; i < K; ++i)
        for (int r = 0; r < m; ++r)
            for (int c = 0; c < m; ++c) {
                cplx wv = w[(long)r * m + c];
                den[obj_index(pos, i, r, c, nr, nc)] += creal(wv) * creal(wv) + cimag(wv) * cimag(wv);
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
#pragma omp parallel for schedule(static)
    for (int r = 0; r < m; ++r)
        for (int c = 0; c < m; ++c) {
            cplx num = 0.0;
            double den = 0.0;
            for (int i = 0; i < K; ++i) {
                cplx pv = psi[obj_index(pos, i, r, c, nr, nc)];
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
                count[obj_index(pos, i, r, c, nr, nc)] += 1;
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

/* Periodic versions of the integer artefacts (reading G25): the index of O10 (i) with the wrap of obj_index(),
 * and the tile lists by brute force over PIXELS: frame i is in tile (ty,tx) iff one of its m x m pixels, taken
 * modulo the image size, falls in the tile.  (Cover counts: orc_cover_counts already goes through obj_index().) */
void orc_linear_index_periodic(int m, int K, const int32_t *pos, int nr, int nc, int64_t *idx)
{
    for (int i = 0; i < K; ++i)
        for (int r = 0; r < m; ++r)
            for (int c = 0; c < m; ++c) idx[((long)i * m + r) * m + c] = (int64_t)obj_index(pos, i, r, c, nr, nc);
}

void orc_tile_lists_periodic(int m, int K, const int32_t *pos, int nr, int nc, int T, int32_t *tile_ptr, int32_t *frames)
{
    int ty_n = (nr + T - 1) / T, tx_n = (nc + T - 1) / T;
    int32_t n = 0;
    for (int ty = 0; ty < ty_n; ++ty)
        for (int tx = 0; tx < tx_n; ++tx) {
            tile_ptr[ty * tx_n + tx] = n;
            for (int i = 0; i < K; ++i) {
                int hit_r = 0, hit_c = 0;
                for (int r = 0; r < m; ++r) if ((pos[2 * i] + r) % nr / T == ty) hit_r = 1;
                for (int c = 0; c < m; ++c) if ((pos[2 * i + 1] + c) % nc / T == tx) hit_c = 1;
                if (hit_r && hit_c) { if (frames) frames[n] = i; ++n; }
            }
        }
    tile_ptr[ty_n * tx_n] = n;
}

/* ------------------------------------------------------------------------------------------------
 * O11 error against a known solution, Eq. (14) PAPER.md:208-212:
 *        eps_0(z) = min_phi || Q*(e^{i phi} z - z_0) || / || Q* z_0 ||,      z_0 = Q psi_0
 *     Q* is the un-normalised overlap sum of O4 ("Notice the additional scaling factor Q*").  Q* uses the
 *     illumination w; z_0 is formed with w0 (the illumination of the known solution; pass w0 = w when the
 *     illumination is given).
 *     With A = Q* z, B = Q* z_0:  || e^{i phi} A - B ||^2 = ||A||^2 + ||B||^2 - 2 Re(e^{i phi} <B, A>), <B,A> = sum conj(B) A,
 *     which is smallest where e^{i phi} <B,A> is real and positive, i.e. phi* = -arg <B,A>.  The oracle takes that
 *     phi* and then EVALUATES the norm of Eq. (14) literally at it (no expanded form); phi_out receives phi*.
 *     tests/test_oracle_next.py checks the minimum against a brute-force scan over phi.
 * ---------------------------------------------------------------------------------------------- */
double orc_eps0(int m, int K, const int32_t *pos, int nr, int nc, const cplx *w, const cplx *w0, const cplx *z,
                const cplx *psi0, double *phi_out)
{
    long N = (long)K * m * m, P = (long)nr * nc;
    cplx *z0 = (cplx *)malloc(sizeof(cplx) * (size_t)N);
    cplx *A = (cplx *)malloc(sizeof(cplx) * (size_t)P);
    cplx *B = (cplx *)malloc(sizeof(cplx) * (size_t)P);
    orc_split(m, K, pos, nr, nc, psi0, w0, z0);
    orc_overlap_num(m, K, pos, nr, nc, w, z, A);
    orc_overlap_num(m, K, pos, nr, nc, w, z0, B);
    cplx ba = 0.0;
    double nb = 0.0;
    for (long p = 0; p < P; ++p) {
        ba += conj(B[p]) * A[p];
        nb += creal(B[p]) * creal(B[p]) + cimag(B[p]) * cimag(B[p]);
    }
    double phi = -carg(ba);
    cplx e = cos(phi) + I * sin(phi);
    double s = 0.0;
    for (long p = 0; p < P; ++p) {
        cplx d = e * A[p] - B[p];
        s += creal(d) * creal(d) + cimag(d) * cimag(d);
    }
    free(z0); free(A); free(B);
    if (phi_out) *phi_out = phi;
    return sqrt(s / nb);
}

/* ------------------------------------------------------------------------------------------------
 * O12 default initialisations, PAPER.md:171-172 (steps 2-3).
 *   step 2  "w0 = inverse Fourier transform of the square root of the average frame":
 *             abar(q) = sqrt( (1/K) sum_i max(I_i(q), 0) ),   w0 = F* abar,
 *           then moved to the frame centre by the cyclic shift (m/2, m/2) (reading G21: abar is real and
 *           non-negative, so F* abar peaks at index (0,0); the illumination lives at the frame centre, PAPER.md:163,
 *           reading G19).
 *   step 3  "psi0 filled with random numbers uniformly drawn from [0,1)": the draw is a counter-based generator
 *           that both sides implement (splitmix64 of seed and pixel index, top 24 bits -> float in [0,1)); real part
 *           = the draw, imaginary part 0.  Compared BIT-EXACTLY with the library.
 * ---------------------------------------------------------------------------------------------- */
void orc_default_probe(int m, int K, const float *Iq, cplx *w0)
{
    long mm = (long)m * m;
    cplx *abar = (cplx *)malloc(sizeof(cplx) * (size_t)mm);
    cplx *t = (cplx *)malloc(sizeof(cplx) * (size_t)mm);
    for (long q = 0; q < mm; ++q) {
        double s = 0.0;
        for (int i = 0; i < K; ++i) {
            double v = (double)Iq[(long)i * mm + q];
            s += (v > 0.0) ? v : 0.0;
        }
        abar[q] = sqrt(s / (double)K);
    }
    orc_fft2(m, abar, t, +1);
    for (int r = 0; r < m; ++r)
        for (int c = 0; c < m; ++c) w0[(long)((r + m / 2) % m) * m + (c + m / 2) % m] = t[(long)r * m + c];
    free(abar); free(t);
}

static uint64_t orc_splitmix64(uint64_t x)
{
    x += 0x9E3779B97F4A7C15ULL;
    uint64_t z = x;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

void orc_random_object(long n, uint64_t seed, float *re)
{
    uint64_t k = orc_splitmix64(seed);
    for (long p = 0; p < n; ++p) re[p] = (float)(orc_splitmix64(k + (uint64_t)p) >> 40) * (1.0f / 16777216.0f);
}

/* ------------------------------------------------------------------------------------------------
 * O13 illumination constraints, step 7 PAPER.md:181-189.
 *   mask:       w <- F^{-1}{ (F w) m_w }                          m_w real (a support: 0/1, or any weights)
 *   amplitude:  w <- F^{-1}{ (F w / |F w|) a_w }                  a_w = |F w_0| >= 0
 *               where |F w| <= thr_w the phase factor is taken as 1, as in G4 (reading G24); the caller passes
 *               thr_w = 1e-4 * rms(a_w).
 *   Both m_w and a_w are indexed like the transform: DC at [0,0].
 * ---------------------------------------------------------------------------------------------- */
void orc_probe_mask(int m, const cplx *w, const double *mask, cplx *out)
{
    long mm = (long)m * m;
    cplx *W = (cplx *)malloc(sizeof(cplx) * (size_t)mm);
    orc_fft2(m, w, W, -1);
    for (long q = 0; q < mm; ++q) W[q] *= mask[q];
    orc_fft2(m, W, out, +1);
    free(W);
}

void orc_probe_amplitude(int m, const cplx *w, const double *aw, double thr_w, cplx *out)
{
    long mm = (long)m * m;
    cplx *W = (cplx *)malloc(sizeof(cplx) * (size_t)mm);
    orc_fft2(m, w, W, -1);
    for (long q = 0; q < mm; ++q) {
        double mag = cabs(W[q]);
        W[q] = (mag > thr_w) ? (W[q] / mag) * aw[q] : (cplx)aw[q];
    }
    orc_fft2(m, W, out, +1);
    free(W);
}

/* ------------------------------------------------------------------------------------------------
 * O14 re-centring, PAPER.md:163 ("keeping the illumination in the center of the frame by computing the center of
 *     mass and correcting for drifts after every update") and :191 ("compute center of mass of w and shift it").
 *     Reading G22: the mass is |w|^2; the centre of mass is the plain first moment over the frame indices,
 *         cm_r = sum r |w(r,c)|^2 / sum |w|^2   (likewise cm_c);
 *     the shift is the INTEGER d = floor(m/2 - cm + 1/2) per axis (positions are integer pixels; the paper
 *     defines no interpolation), applied cyclically: w'(r) = w((r - d) mod m).  Only w moves (reading G23).
 *     d_out receives (d_r, d_c).  With sum |w|^2 = 0 nothing moves.
 * ---------------------------------------------------------------------------------------------- */
void orc_probe_recentre(int m, const cplx *w, cplx *out, int32_t d_out[2])
{
    double s = 0.0, sr = 0.0, sc = 0.0;
    for (int r = 0; r < m; ++r)
        for (int c = 0; c < m; ++c) {
            cplx v = w[(long)r * m + c];
            double p = creal(v) * creal(v) + cimag(v) * cimag(v);
            s += p; sr += p * r; sc += p * c;
        }
    int dr = 0, dc = 0;
    if (s > 0.0) {
        dr = (int)floor((double)(m / 2) - sr / s + 0.5);
        dc = (int)floor((double)(m / 2) - sc / s + 0.5);
    }
    for (int r = 0; r < m; ++r)
        for (int c = 0; c < m; ++c)
            out[(long)(((r + dr) % m + m) % m) * m + ((c + dc) % m + m) % m] = w[(long)r * m + c];
    d_out[0] = dr; d_out[1] = dc;
}
