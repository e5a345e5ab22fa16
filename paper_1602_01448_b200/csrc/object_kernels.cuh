// object_kernels.cuh -- everything that is not the fused FFT kernel: split (a1), the deterministic gather-form
// overlap with its object-space epilogues (a5 + the object half of a6), the illumination refinement (a7), the
// amplitude preparation (a0) and small helpers.
#pragma once
#include "frame_common.cuh"
#include "frame_r.cuh"
#include "frame_s.cuh"

namespace sharp {

constexpr int TILE = 32;  // == SHARP_TILE

// T_i: linear object index under frame pixel (r, c) of a frame at (xr, xc).  With the periodic boundary of the Fig. 3
// simulation (reading G25) positions lie anywhere in the image and r + x_i is taken modulo its size;
// for the positions of PAPER.md:53 (x_i <= n - m) the two corrections never fire.
__device__ __forceinline__ size_t obj_index(int xr, int xc, int r, int c, int nr, int nc)
{
    int rr = xr + r, cc = xc + c;
    if (rr >= nr) rr -= nr;
    if (cc >= nc) cc -= nc;
    return (size_t)rr * nc + cc;
}

// ---------------------------------------------------------------------------------------------------------
// a1 split:  z_i(r) = w(r) psi(r + x_i).  One thread per two consecutive frame pixels of a
// row: 128-bit loads of w and stores of z; psi is only 8-byte aligned (x_i.col is arbitrary) so it is read as
// two 64-bit loads.  psi == NULL means the flat object 1 + 0i (reading G8).
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_split(int m, int K, const int *pos, int nr, int nc, const float2 *psi,
                                                const float2 *w, float2 *z)
{
    const size_t half = (size_t)m / 2;
    const size_t per_frame = (size_t)m * half;
    const size_t total = (size_t)K * per_frame;
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(g / per_frame);
        const size_t rem = g - (size_t)i * per_frame;
        const int r = (int)(rem / half), c = 2 * (int)(rem % half);
        const float4 w2 = __ldg(reinterpret_cast<const float4 *>(w + (size_t)r * m + c));
        float2 p0 = make_float2(1.f, 0.f), p1 = p0;
        if (psi != nullptr) {
            p0 = __ldg(psi + obj_index(pos[2 * i], pos[2 * i + 1], r, c, nr, nc));
            p1 = __ldg(psi + obj_index(pos[2 * i], pos[2 * i + 1], r, c + 1, nr, nc));
        }
        const float2 z0 = cmul(make_float2(w2.x, w2.y), p0), z1 = cmul(make_float2(w2.z, w2.w), p1);
        __stcs(reinterpret_cast<float4 *>(z + ((size_t)i * m + r) * m + c), make_float4(z0.x, z0.y, z1.x, z1.y));
    }
}

// z = c + w_form . T psi_v  (materialise the frames kept in factored form; sharp_get_frames)
__global__ void __launch_bounds__(256) k_materialize(int m, int K, const int *pos, int nr, int nc, const float2 *c,
                                                      const float2 *psi_v, const float2 *w, float2 *z)
{
    const size_t per_frame = (size_t)m * m;
    const size_t total = (size_t)K * per_frame;
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(g / per_frame);
        const size_t rem = g - (size_t)i * per_frame;
        const int r = (int)(rem / m), col = (int)(rem % m);
        float2 v = __ldcs(c + g);
        if (psi_v != nullptr)
            v = cadd(v, cmul(__ldg(w + rem), __ldg(psi_v + obj_index(pos[2 * i], pos[2 * i + 1], r, col, nr, nc))));
        z[g] = v;
    }
}

// linear object index of frame pixel (i, r, c), with the same expression the kernels above use (O10 (i))
__global__ void __launch_bounds__(256) k_frame_index(int m, int K, const int *pos, int nr, int nc, long long *idx)
{
    const size_t per_frame = (size_t)m * m;
    const size_t total = (size_t)K * per_frame;
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(g / per_frame);
        const size_t rem = g - (size_t)i * per_frame;
        const int r = (int)(rem / m), col = (int)(rem % m);
        idx[g] = (long long)obj_index(pos[2 * i], pos[2 * i + 1], r, col, nr, nc);
    }
}

// ---------------------------------------------------------------------------------------------------------
// a0 amplitudes:  a = sqrt(max(I, 0))  (reading G14), stored as a/m in the order in which the frame
// kernel of this frame size meets the Fourier coefficients ("slots"): slot_freq() of frame_r.cuh for m <= 128,
// slot_freq_s() of frame_s.cuh above.
// Also per-block partial sums of max(I,0) in double (||a||^2, reading G12); k_scalars finishes them in a fixed
// order.  k_amplitudes_natural is the inverse map (a_int -> a, for sharp_get_amplitudes).
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void amp_slot_freq(int m, int slot, int &u, int &v)
{
    if (m == 64) slot_freq<64>(slot, u, v);
    else if (m == 128) slot_freq<128>(slot, u, v);
    else if (m == 256) slot_freq_s<256>(slot, u, v);
    else slot_freq_s<512>(slot, u, v);
}

__global__ void __launch_bounds__(256) k_amplitudes(int m, int K, const float *I, float *a_int,
                                                     double *partials)
{
    const size_t per_frame = (size_t)m * m;
    const size_t total = (size_t)K * per_frame;
    const float inv_m = 1.0f / (float)m;
    double acc = 0.0;
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (size_t)gridDim.x * blockDim.x) {
        const size_t i = g / per_frame;
        int u, v;
        amp_slot_freq(m, (int)(g - i * per_frame), u, v);
        const float val = fmaxf(__ldg(I + i * per_frame + (size_t)u * m + v), 0.0f);
        acc += (double)val;
        a_int[g] = sqrtf(val) * inv_m;
    }
    __shared__ double red[256];
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int off = 128; off > 0; off >>= 1) {
        if ((int)threadIdx.x < off) red[threadIdx.x] += red[threadIdx.x + off];
        __syncthreads();
    }
    if (threadIdx.x == 0) partials[blockIdx.x] = red[0];
}

__global__ void k_amplitudes_natural(int m, int K, const float *a_int, float *a)
{
    const size_t per_frame = (size_t)m * m;
    const size_t total = (size_t)K * per_frame;
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (size_t)gridDim.x * blockDim.x) {
        const size_t i = g / per_frame;
        int u, v;
        amp_slot_freq(m, (int)(g - i * per_frame), u, v);
        a[i * per_frame + (size_t)u * m + v] = a_int[g] * (float)m;
    }
}

// A2 = sum of the partials in index order; thr2 = (m thr)^2 = tau^2 A2 / K  with thr = tau a_rms (reading G4).
__global__ void k_scalars(int nparts, const double *partials, int K, double tau, DevScalars *sc)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double s = 0.0;
        for (int j = 0; j < nparts; ++j) s += partials[j];
        sc->A2 = s;
        sc->thr2 = (float)(tau * tau * s / (double)K);
        sc->pad = 0.f;
    }
}

// sharded plan: A2 has been summed over the ranks; thr2 follows from the global mean (K_total frames)
__global__ void k_scalars_thr(long long K_total, double tau, DevScalars *sc)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) sc->thr2 = (float)(tau * tau * sc->A2 / (double)K_total);
}

// sums gridDim-many triples in index order into out[3] (eps numerators, doubles)
__global__ void k_sum_triples(int n, const double *partials, double *out)
{
    if (threadIdx.x < 3 && blockIdx.x == 0) {
        double s = 0.0;
        for (int j = 0; j < n; ++j) s += partials[3 * j + threadIdx.x];
        out[threadIdx.x] = s;
    }
}

// ---------------------------------------------------------------------------------------------------------
// a5 overlap, gather form (PAPER.md:153-155 Eq. 9; :224 "the image is divided into blocks ... each block
// determines which frames contribute").  One CTA per TILE x TILE object tile; the tile's CSR list gives the
// frames that touch it, in ascending frame index, so every pixel's sum runs in ascending i with no atomics
// (reading G17).  256 threads, each owning one column and four rows (ty, ty+8, ty+16, ty+24) of the tile.
//
//   num(p)   = sum_i conj(w_a(p - x_i)) f_i(p - x_i)
//   cross(p) = sum_i conj(w_a(p - x_i)) w_b(p - x_i)            (OV_DEN with w_b given: kept for OV_REGATHER)
//   den(p)   = sum_i |w_a(p - x_i)|^2                            (OV_DEN only; otherwise read from the den array)
// Epilogues:
//   OV_DEN       den[p] = sum |w_a|^2;  cross[p] = sum conj(w_a) w_b when w_b is given (no frame data touched)
//   OV_L         out[p] = num/den, 0 where den == 0 (reading G5)
//   OV_ITER      psi_c = num/den; psi_y = (psi_c - beta psi_z)/(1 - 2 beta); psi_v[p] = beta (2 psi_y - psi_z);
//                psi_z[p] = psi_y                                (object half of RAAR)
//   OV_REGATHER  psi_z[p] = (num + psi_v[p] cross[p])/den        (L_{w_a}(c + w_b . T psi_v) after w changed)
//   OV_BLIND     the iteration that follows an illumination update, in ONE pass: with w_a the new illumination, w_b the
//                one the frames z = f_prev + w_b . T psi_v_in were formed with, and f the new frame-local state c'':
//                den = sum |w_a|^2, cross = sum conj(w_a) w_b, n0 = sum conj(w_a) f_prev, n1 = sum conj(w_a) f;
//                psi_z = (n0 + psi_v_in cross)/den  (= L_{w_a} z, what OV_DEN + OV_REGATHER would have produced), then the
//                OV_ITER epilogue on n1/den with that psi_z; den[p] is written for later use.
// ---------------------------------------------------------------------------------------------------------
enum OverlapMode : int { OV_DEN = 0, OV_L = 1, OV_ITER = 2, OV_REGATHER = 3, OV_BLIND = 4 };

struct OverlapArgs {
    int m, nr, nc, tiles_c;
    int periodic;           // positions anywhere in the image, frames wrap around its edges (reading G25)
    const int *pos;
    const int *tile_ptr;
    const int *tile_frames;
    const float2 *f;        // K m m
    const float2 *f_prev;   // K m m (OV_BLIND: the state the current frames were formed from)
    const float2 *w_a;      // m m
    const float2 *w_b;      // m m (DEN: second probe of the cross term, may be NULL)
    float2 *cross;          // object-sized (DEN out when w_b given, REGATHER in)
    float *den;             // object-sized
    float2 *out;            // OV_L
    float2 *psi_z;          // ITER in/out, REGATHER out
    const float2 *psi_v_in; // REGATHER
    float2 *psi_v_out;      // ITER
    float2 *num_out;        // not NULL: write the raw numerator here and skip the epilogue (sharded plan)
    float beta;
};

// Object-space epilogue of one pixel p with numerator num(p) (written once; the gather kernel and the sharded
// two-step path both end here):
//   OV_L         out[p] = num/den, 0 where den == 0 (reading G5)
//   OV_ITER      psi_c = num/den; psi_y = (psi_c - beta psi_z)/(1 - 2 beta); psi_v[p] = beta (2 psi_y - psi_z); psi_z[p] = psi_y
//   OV_REGATHER  psi_z[p] = (num + psi_v[p] cross[p])/den
template <int MODE>
__device__ __forceinline__ void object_epilogue(const OverlapArgs &A, size_t p, float2 num)
{
    const float d = A.den[p];
    const bool lit = d > 0.f;
    if constexpr (MODE == OV_L) {
        A.out[p] = lit ? make_float2(num.x / d, num.y / d) : make_float2(0.f, 0.f);
    } else if constexpr (MODE == OV_ITER) {
        float2 py = make_float2(0.f, 0.f), pv = py;
        if (lit) {
            const float2 pz = A.psi_z[p];
            const float inv = 1.0f / (1.0f - 2.0f * A.beta);
            py.x = (num.x / d - A.beta * pz.x) * inv;
            py.y = (num.y / d - A.beta * pz.y) * inv;
            pv.x = A.beta * (2.0f * py.x - pz.x);
            pv.y = A.beta * (2.0f * py.y - pz.y);
        }
        A.psi_z[p] = py;
        A.psi_v_out[p] = pv;
    } else {  // OV_REGATHER
        float2 o = make_float2(0.f, 0.f);
        if (lit) {
            float2 t = num;
            if (A.psi_v_in != nullptr) t = cadd(t, cmul(A.psi_v_in[p], A.cross[p]));
            o = make_float2(t.x / d, t.y / d);
        }
        A.psi_z[p] = o;
    }
}

// The gather loop.  M is a template parameter so that the four rows of a thread are immediate offsets from one pointer
// per array.  The tile's list is staged in shared memory in chunks of CH entries as, per frame: the element offset of
// the tile's corner pixel inside the frame data and inside the probe (so a thread's address is that plus its own
// constant ty M + tx), and the range of tile rows / columns the frame covers, packed in one word.  UNR frames are in
// flight per thread at a time and are accumulated in list order (ascending frame index: reading G17).
#ifndef SHARP_OV_UNR
#define SHARP_OV_UNR 3
#endif
#ifndef SHARP_OVB_UNR          // OV_BLIND: four arrays per (frame, row) pair
#define SHARP_OVB_UNR 1
#endif
#ifndef SHARP_OVB_MINB
#define SHARP_OVB_MINB 3
#endif
#ifndef SHARP_OV_MINB
#define SHARP_OV_MINB 4
#endif
// Two things decide how many loads ptxas (12.9) keeps in flight here, and both were found the hard way:
//  - with __launch_bounds__(256) alone it allocates 39 registers and interleaves every pair of loads with the arithmetic that
//    consumes it; with a minimum CTA count given it batches the loads as written;
//  - arithmetic predicated with the same condition as its loads keeps one of the 7 predicate registers live per (frame, row)
//    pair, which caps a batch at 6-7 pairs; out-of-range pairs are therefore loaded as zeros and accumulated unconditionally.
// Measured at config 2 (us per launch; UNR frames per batch / minimum CTAs): predicated 4/3 104.6, 6/2 101.1; unconditional
// 4/2 123, 6/2 118, 4/3 99.1, 2/4 94.5, 2/5 94.6, 3/4 91.6 (kept), 3/5 132, 2/6 112, 1/8 117: occupancy (32 warps) buys more
// than a longer batch per thread.  OV_BLIND (config 3): 2/2 176.8, 1/3 170.6 (kept), 1/4 169.0, 2/3 232, 1/2 215.
template <int M, int MODE>
__global__ void __launch_bounds__(256, MODE == OV_BLIND ? SHARP_OVB_MINB : SHARP_OV_MINB) k_overlap(OverlapArgs A)
{
    const int tile = blockIdx.x;
    const int tr = tile / A.tiles_c, tc = tile % A.tiles_c;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int pc = tc * TILE + tx;
    const int pr0 = tr * TILE + ty;
    const int beg = A.tile_ptr[tile], end = A.tile_ptr[tile + 1];
    const int toff = ty * M + tx;

    float2 num[4], cr[4], n0[4];
    float dn[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        num[k] = make_float2(0.f, 0.f);
        cr[k] = make_float2(0.f, 0.f);
        n0[k] = make_float2(0.f, 0.f);
        dn[k] = 0.f;
    }

    constexpr int CH = 128, UNR = (MODE == OV_BLIND) ? SHARP_OVB_UNR : SHARP_OV_UNR;
    __shared__ long long s_foff[CH];     // fi M^2 + (tile row0 - x_r) M + (tile col0 - x_c): may be negative before toff is added
    __shared__ int s_woff[CH];           // the same without the frame term
    __shared__ unsigned s_rng[CH];       // r_lo | r_hi << 8 | c_lo << 16 | c_hi << 24  (tile-local, half-open)
    for (int base = beg; base < end; base += CH) {
        const int n = min(CH, end - base);
        __syncthreads();
        for (int j = threadIdx.x; j < n; j += blockDim.x) {
            const int fi = __ldg(A.tile_frames + base + j);
            int xr = __ldg(A.pos + 2 * fi), xc = __ldg(A.pos + 2 * fi + 1);
            if (A.periodic) {
                // the copy of the frame (at x or at x - n) that meets this tile: a frame that starts beyond the tile
                // reaches it by wrapping (the plan guarantees n - m >= TILE - 1, so never both)
                if (xr > tr * TILE + TILE - 1) xr -= A.nr;
                if (xc > tc * TILE + TILE - 1) xc -= A.nc;
            }
            const int dr = tr * TILE - xr, dc = tc * TILE - xc;          // frame coordinates of the tile's corner
            const int wo = dr * M + dc;
            s_woff[j] = wo;
            s_foff[j] = (long long)fi * (M * M) + wo;
            const int rlo = max(0, -dr), rhi = min(TILE, M - dr), clo = max(0, -dc), chi = min(TILE, M - dc);
            s_rng[j] = (unsigned)rlo | ((unsigned)rhi << 8) | ((unsigned)clo << 16) | ((unsigned)chi << 24);
        }
        __syncthreads();
        for (int e0 = 0; e0 < n; e0 += UNR) {
            float2 fv[UNR][4], wa[UNR][4], wb[UNR][4], fp0[UNR][4];
            bool ok[UNR][4];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const int e = min(e0 + u, n - 1);
                const unsigned rng = s_rng[e];
                const int rlo = rng & 255, rh = ((rng >> 8) & 255) - rlo, clo = (rng >> 16) & 255, cw = (rng >> 24) - clo;
                const bool colok = (e0 + u < n) && ((unsigned)(tx - clo) < (unsigned)cw);
                const int wo = s_woff[e] + toff;
                const float2 *wp = A.w_a + wo;
                const float2 *fp = (MODE == OV_DEN) ? nullptr : A.f + (s_foff[e] + toff);
                const float2 *bp = (MODE == OV_BLIND || (MODE == OV_DEN && A.w_b != nullptr)) ? A.w_b + wo : nullptr;
                const float2 *qp = (MODE == OV_BLIND) ? A.f_prev + (s_foff[e] + toff) : nullptr;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    ok[u][k] = colok && ((unsigned)(ty + 8 * k - rlo) < (unsigned)rh);
                    wa[u][k] = make_float2(0.f, 0.f);
                    fv[u][k] = make_float2(0.f, 0.f);
                    wb[u][k] = make_float2(0.f, 0.f);
                    fp0[u][k] = make_float2(0.f, 0.f);
                    if (ok[u][k]) {
                        wa[u][k] = __ldg(wp + 8 * k * M);
                        if constexpr (MODE != OV_DEN) fv[u][k] = __ldcs(fp + 8 * k * M);
                        if constexpr (MODE == OV_DEN) { if (bp != nullptr) wb[u][k] = __ldg(bp + 8 * k * M); }
                        if constexpr (MODE == OV_BLIND) {
                            wb[u][k] = __ldg(bp + 8 * k * M);
                            fp0[u][k] = __ldcs(qp + 8 * k * M);
                        }
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    // unconditional: a pair that is out of range was loaded as w = f = 0 and adds nothing.  (Predicating the
                    // arithmetic as well keeps one of the 7 predicate registers live per pair from the load to its use, which
                    // caps the loads ptxas can batch at 6-7 pairs.)
                    const float2 w_ = wa[u][k];
                    if constexpr (MODE == OV_DEN) {
                        dn[k] += w_.x * w_.x + w_.y * w_.y;
                        const float2 b_ = wb[u][k];
                        cr[k].x += w_.x * b_.x + w_.y * b_.y;     // conj(w_a) w_b (zero when w_b is absent)
                        cr[k].y += w_.x * b_.y - w_.y * b_.x;
                    } else {
                        const float2 f_ = fv[u][k];
                        num[k].x += w_.x * f_.x + w_.y * f_.y;   // conj(w_a) f
                        num[k].y += w_.x * f_.y - w_.y * f_.x;
                        if constexpr (MODE == OV_BLIND) {
                            const float2 b_ = wb[u][k], q_ = fp0[u][k];
                            dn[k] += w_.x * w_.x + w_.y * w_.y;
                            cr[k].x += w_.x * b_.x + w_.y * b_.y;
                            cr[k].y += w_.x * b_.y - w_.y * b_.x;
                            n0[k].x += w_.x * q_.x + w_.y * q_.y;
                            n0[k].y += w_.x * q_.y - w_.y * q_.x;
                        }
                    }
                }
            }
        }
    }

    if (pc >= A.nc) return;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int pr = pr0 + 8 * k;
        if (pr >= A.nr) continue;
        const size_t p = (size_t)pr * A.nc + pc;
        if constexpr (MODE == OV_DEN) {
            A.den[p] = dn[k];
            if (A.w_b != nullptr) A.cross[p] = cr[k];
        } else if constexpr (MODE == OV_BLIND) {
            const float d = dn[k];
            A.den[p] = d;
            float2 pz = make_float2(0.f, 0.f), py = pz, pv = pz;
            if (d > 0.f) {
                float2 t = n0[k];
                if (A.psi_v_in != nullptr) t = cadd(t, cmul(A.psi_v_in[p], cr[k]));
                pz = make_float2(t.x / d, t.y / d);                     // L_{w_a} z: the re-gathered estimate
                const float inv = 1.0f / (1.0f - 2.0f * A.beta);
                py.x = (num[k].x / d - A.beta * pz.x) * inv;
                py.y = (num[k].y / d - A.beta * pz.y) * inv;
                pv.x = A.beta * (2.0f * py.x - pz.x);
                pv.y = A.beta * (2.0f * py.y - pz.y);
            }
            A.psi_z[p] = py;
            A.psi_v_out[p] = pv;
        } else {
            if (A.num_out != nullptr) A.num_out[p] = num[k];     // sharded plan: the sum over ranks comes first
            else object_epilogue<MODE>(A, p, num[k]);
        }
    }
}

// The object-space epilogue alone, on a numerator that was summed over the ranks of a sharded reconstruction
// ("the resulting image is summed across all MPI nodes").
template <int MODE>
__global__ void __launch_bounds__(256) k_object_epilogue(OverlapArgs A, const float2 *num)
{
    const size_t n = (size_t)A.nr * A.nc;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (size_t)gridDim.x * blockDim.x)
        object_epilogue<MODE>(A, p, num[p]);
}

// ---------------------------------------------------------------------------------------------------------
// a7 illumination refinement, Eq. (10) PAPER.md:157-159:
//     w(r) <- sum_i conj(psi(r + x_i)) z_i(r) / sum_i |psi(r + x_i)|^2
// with z_i = c_i + w_form . T psi_v formed on the fly.  Two stages, both in a fixed order: each CTA column sums
// a chunk of consecutive frames (ascending i) per probe pixel; k_probe_final adds the chunks in ascending order
// and divides; where the denominator is 0 the old value is kept.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_probe_partial(int m, int K, int chunk, const int *pos, int nr, int nc,
                                                        const float2 *c, const float2 *psi_v, const float2 *w_form,
                                                        const float2 *psi, float2 *pnum, float *pden)
{
    // one frame in flight per thread at 32 registers and full occupancy: measured 87 us at config 3; four frames in
    // flight with the chunk's positions staged in shared memory (55 registers, half the warps) 94 us
    const int pix = blockIdx.x * blockDim.x + threadIdx.x;  // m*m is a multiple of 256
    const int r = pix / m, col = pix % m;
    const int i0 = blockIdx.y * chunk, i1 = min(K, i0 + chunk);
    const float2 wf = __ldg(w_form + pix);
    float2 num = make_float2(0.f, 0.f);
    float den = 0.f;
    for (int i = i0; i < i1; ++i) {
        const size_t op = obj_index(__ldg(pos + 2 * i), __ldg(pos + 2 * i + 1), r, col, nr, nc);
        const float2 ps = __ldg(psi + op);
        float2 z = __ldcs(c + (size_t)i * m * m + pix);
        if (psi_v != nullptr) z = cadd(z, cmul(wf, __ldg(psi_v + op)));
        num.x += ps.x * z.x + ps.y * z.y;  // conj(ps) * z
        num.y += ps.x * z.y - ps.y * z.x;
        den += ps.x * ps.x + ps.y * ps.y;
    }
    pnum[(size_t)blockIdx.y * m * m + pix] = num;
    pden[(size_t)blockIdx.y * m * m + pix] = den;
}

// raw != NULL (sharded plan): the sums (num.x, num.y, den) go to raw[3 pix ..] for the sum over ranks and
// k_probe_divide finishes
__global__ void __launch_bounds__(256) k_probe_final(int m, int nchunks, const float2 *pnum, const float *pden,
                                                      const float2 *w_old, float2 *w_new, float *raw)
{
    const int pix = blockIdx.x * blockDim.x + threadIdx.x;
    float2 num = make_float2(0.f, 0.f);
    float den = 0.f;
    for (int j = 0; j < nchunks; ++j) {
        const float2 a = pnum[(size_t)j * m * m + pix];
        num.x += a.x;
        num.y += a.y;
        den += pden[(size_t)j * m * m + pix];
    }
    if (raw != nullptr) {
        raw[3 * pix + 0] = num.x;
        raw[3 * pix + 1] = num.y;
        raw[3 * pix + 2] = den;
        return;
    }
    w_new[pix] = den > 0.f ? make_float2(num.x / den, num.y / den) : w_old[pix];
}

__global__ void __launch_bounds__(256) k_probe_divide(const float *raw, const float2 *w_old, float2 *w_new)
{
    const int pix = blockIdx.x * blockDim.x + threadIdx.x;
    const float den = raw[3 * pix + 2];
    w_new[pix] = den > 0.f ? make_float2(raw[3 * pix] / den, raw[3 * pix + 1] / den) : w_old[pix];
}

__global__ void k_fill_c64(size_t n, float2 *p, float2 v)
{
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < n; g += (size_t)gridDim.x * blockDim.x) p[g] = v;
}

}  // namespace sharp
