// frame_kernel.cuh -- the fused per-frame kernel: form z, 2-D FFT, Fourier-magnitude projection folded with
// the RAAR frame-local combination, inverse 2-D FFT (steps a1-a4 and the frame-local half of a6 in DESIGN.md).
//
// What one frame goes through (PAPER.md:141-143 Eq. 7, :174-178 step 5):
//     z  = c_prev + w_form . T_i psi_v                     (psi_v = beta (2 psi_y - psi_z), the overlap kernel's output)
//     Z^ = FFT2_unnormalised(z)                             (= m * F z, F the unitary DFT of Eq. 2)
//     C^ = Z^ * (beta/m^2 + (1-2 beta) (a/m) / |Z^|)        (|F z| > thr; else C^ = beta/m^2 Z^ + (1-2 beta) a/m: reading G4)
//     c  = IFFT2_unnormalised(C^) = beta z + (1 - 2 beta) P_a z
// so the frame never leaves the SM's reach between F and F*: the row pass exchanges through shared memory and
// the row<->column transposition goes through a per-CTA scratch that lives in L2.
//
// 1-D transform of length M = RA * RB, two in-place passes (DIF forward, DIT inverse, mirrored so that no
// reordering is ever needed):
//   position n = RB n1 + n2  --pass A: DFT_RA over n1, x W_M^{n2 k1}-->  position RB k1 + n2
//                            --pass B: DFT_RB over n2               -->  position RB k1 + k2  holds frequency k1 + RA k2
// The Fourier-domain data therefore sit in "position space"; the amplitudes are stored pre-permuted into that
// space (a_int[q][p] = a[freq(q)][freq(p)] / m, freq(x) = x / RB + RA (x % RB)), see k_amplitudes.
//
// Thread mappings inside a strip of L lines (a line = one row, or one column held as a row of the transposed
// scratch):
//   A-type: thread = (line = tid / TPL, s = tid % TPL) holds positions s + j TPL, j < E   (strided; lanes along
//           the line: coalesced global rows, conflict-free 64-bit shared accesses)
//   B-type: thread = (line = tid % L, t = tid / L) holds positions E t .. E t + E-1        (contiguous; lanes across
//           lines: coalesced accesses of the TRANSPOSED scratch, conflict-free 128-bit shared accesses)
// Shared strip layout: element (line, pos) at line * M + (pos ^ (bitrev3(line & 7) << 1)).
#pragma once
#include "fft_regs.cuh"
#include "frame_common.cuh"

namespace sharp {

template <int M, int E, int NT>
struct FrameCfg {
    static constexpr int RA = E, RB = M / E, TPL = M / E, L = E * NT / M, NSTRIP = M / L;
    static constexpr int SMEM_BYTES = E * NT * 8;
    static_assert(M % E == 0 && (E * NT) % M == 0 && M % L == 0, "bad frame configuration");
    static_assert(L >= 8 || M == 512, "strip too thin");
};

__device__ __forceinline__ int swz(int line, int pos) { return pos ^ ((__brev((unsigned)(line & 7)) >> 29) << 1); }

// A-side twiddles W_M^{k s} (k < E), conjugated for the inverse.  E == 16: per-thread registers; otherwise a
// shared table of M entries.
template <int M, int E>
struct Twiddles {
    static constexpr bool IN_REGS = (E <= 16);
    float2 r[IN_REGS ? E : 1];
    const float2 *tab;
    int s;
    __device__ __forceinline__ void init(float2 *smem_tab, int s_, int tid, int nt)
    {
        s = s_;
        tab = smem_tab;
        if constexpr (IN_REGS) {
#pragma unroll
            for (int k = 0; k < E; ++k) {
                float sn, cs;
                sincospif(-2.0f * (float)(k * s) / (float)M, &sn, &cs);
                r[k] = make_float2(cs, sn);
            }
        } else {
            for (int idx = tid; idx < M; idx += nt) {
                float sn, cs;
                sincospif(-2.0f * (float)idx / (float)M, &sn, &cs);
                smem_tab[idx] = make_float2(cs, sn);
            }
            __syncthreads();
        }
    }
    __device__ __forceinline__ float2 get(int k) const
    {
        if constexpr (IN_REGS) return r[k];
        else return tab[k * s];
    }
};

template <int E, int RB, int SGN>
__device__ __forceinline__ void dft_b(float2 *v)
{
#pragma unroll
    for (int q = 0; q < E / RB; ++q) dft<RB, SGN>(v + q * RB);
}

// Launched with cluster dimension CS (CS = 1: plain launch).  gridDim.x is a multiple of CS.
template <int M, int E, int NT, int MODE, int CS>
__global__ void __launch_bounds__(NT, 2) k_frame(FrameArgs A)
{
    using C = FrameCfg<M, E, NT>;
    constexpr int TPL = C::TPL, L = C::L, RB = C::RB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *strip = reinterpret_cast<float2 *>(smem_raw);
    float2 *tw_tab = strip + E * NT;  // only allocated when E > 16

    const int tid = threadIdx.x;
    const int lineA = tid / TPL, s = tid % TPL;  // A-type
    const int lineB = tid % L, t = tid / L;      // B-type
    const int swzA = (int)((__brev((unsigned)(lineA & 7)) >> 29) << 1);
    const int swzB = (int)((__brev((unsigned)(lineB & 7)) >> 29) << 1);

    Twiddles<M, E> tw;
    tw.init(tw_tab, s, tid, NT);

    const int crank = CS > 1 ? (int)cluster_rank() : 0;
    const int cid = blockIdx.x / CS, nclusters = gridDim.x / CS;
    float2 *scr = A.scratch + (size_t)cid * M * M;
    static_assert(C::NSTRIP % CS == 0, "strips must divide evenly over the cluster");
    const float thr2 = A.sc->thr2;
    const float bm = A.bm, om = A.om;
    double e_a = 0.0, e_q = 0.0, e_d = 0.0;

    for (int i = cid; i < A.K; i += nclusters) {
        const int xr = A.pos[2 * i], xc = A.pos[2 * i + 1];
        const size_t fbase = (size_t)i * M * M;
        // the cluster's next frame (state and amplitudes) is pulled into L2 while this one is transformed
        if (tid == 0 && crank == 0 && i + nclusters < A.K) {
            const size_t nb = (size_t)(i + nclusters) * M * M;
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(A.c_in + nb), "r"(M * M * 8) : "memory");
            if (MODE != FRAME_FFT)
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(A.a_int + nb), "r"(M * M * 4) : "memory");
        }

        // ---------------- stage 1: rows.  form z, pass A, exchange, pass B, store transposed -------------
        for (int sp = crank; sp < C::NSTRIP; sp += CS) {
            const int r0 = sp * L;
            float2 v[E];
            {
                const int r = r0 + lineA;
                const float2 *cin = A.c_in + fbase + (size_t)r * M;
#pragma unroll
                for (int j = 0; j < E; ++j) v[j] = ld_stream(cin + s + j * TPL);
                if (MODE == FRAME_FFT && A.conj_io) {
#pragma unroll
                    for (int j = 0; j < E; ++j) v[j].y = -v[j].y;
                }
                if (A.psi_v != nullptr) {
                    const float2 *wrow = A.w_form + r * M;
                    const float2 *prow = A.psi_v + (size_t)(xr + r) * A.nc + xc;
#pragma unroll
                    for (int j = 0; j < E; ++j) {
                        const int col = s + j * TPL;
                        v[j] = cadd(v[j], cmul(__ldg(wrow + col), __ldg(prow + col)));
                    }
                }
                if constexpr (MODE == FRAME_ERR) {
                    const float2 *wc = A.w_cur + r * M;
                    const float2 *pz = A.psi_z + (size_t)(xr + r) * A.nc + xc;
                    float sq = 0.f, sd = 0.f;
#pragma unroll
                    for (int j = 0; j < E; ++j) {
                        const int col = s + j * TPL;
                        float2 d = csub(cmul(__ldg(wc + col), __ldg(pz + col)), v[j]);
                        sq += d.x * d.x + d.y * d.y;
                        float2 zp = make_float2(0.f, 0.f);
                        if (A.c_prev != nullptr) {
                            zp = ld_stream(A.c_prev + fbase + (size_t)r * M + col);
                            if (A.psi_v_prev != nullptr)
                                zp = cadd(zp, cmul(__ldg(A.w_form_prev + r * M + col),
                                                   __ldg(A.psi_v_prev + (size_t)(xr + r) * A.nc + xc + col)));
                        }
                        float2 dd = csub(v[j], zp);
                        sd += dd.x * dd.x + dd.y * dd.y;
                    }
                    e_q += (double)sq;
                    e_d += (double)sd;
                }
                dft<E, -1>(v);
#pragma unroll
                for (int k = 1; k < E; ++k) v[k] = cmul(v[k], tw.get(k));
                float2 *row = strip + lineA * M;
#pragma unroll
                for (int k = 0; k < E; ++k) row[(s + k * TPL) ^ swzA] = v[k];
            }
            __syncthreads();
            {
                const float4 *row4 = reinterpret_cast<const float4 *>(strip + lineB * M);
#pragma unroll
                for (int jj = 0; jj < E; jj += 2) {
                    float4 q4 = row4[((E * t + jj) ^ swzB) >> 1];
                    v[jj] = make_float2(q4.x, q4.y);
                    v[jj + 1] = make_float2(q4.z, q4.w);
                }
                dft_b<E, RB, -1>(v);
                float2 *dst = scr + (size_t)(E * t) * M + (r0 + lineB);
#pragma unroll
                for (int jj = 0; jj < E; ++jj) st_l2(dst + (size_t)jj * M, v[jj]);
            }
            __syncthreads();
        }

        if (CS > 1) cluster_barrier();
        // ---------------- stage 2: columns (rows of the transposed scratch).  A, B, project, B^-1, A^-1 ----
        for (int sp = crank; sp < C::NSTRIP; sp += CS) {
            const int p0 = sp * L;
            float2 v[E];
            {
                const float2 *src = scr + (size_t)(p0 + lineA) * M;
#pragma unroll
                for (int j = 0; j < E; ++j) v[j] = ld_l2(src + s + j * TPL);
                dft<E, -1>(v);
#pragma unroll
                for (int k = 1; k < E; ++k) v[k] = cmul(v[k], tw.get(k));
                float2 *row = strip + lineA * M;
#pragma unroll
                for (int k = 0; k < E; ++k) row[(s + k * TPL) ^ swzA] = v[k];
            }
            __syncthreads();
            {
                float4 *row4 = reinterpret_cast<float4 *>(strip + lineB * M);
#pragma unroll
                for (int jj = 0; jj < E; jj += 2) {
                    float4 q4 = row4[((E * t + jj) ^ swzB) >> 1];
                    v[jj] = make_float2(q4.x, q4.y);
                    v[jj + 1] = make_float2(q4.z, q4.w);
                }
                dft_b<E, RB, -1>(v);
                // v[jj] = Z^ at (q = E t + jj, p = p0 + lineB) in position space
                const int p = p0 + lineB;
                if constexpr (MODE == FRAME_FFT) {
                    // natural-order, unitary output (test hook): frequency of a position x is x / RB + RA (x % RB)
                    const int vfreq = p / RB + C::RA * (p % RB);
                    const float inv_m = 1.0f / (float)M;
#pragma unroll
                    for (int jj = 0; jj < E; ++jj) {
                        const int q = E * t + jj;
                        const int ufreq = q / RB + C::RA * (q % RB);
                        float2 o = make_float2(v[jj].x * inv_m, v[jj].y * inv_m);
                        if (A.conj_io) o.y = -o.y;
                        A.c_out[fbase + (size_t)ufreq * M + vfreq] = o;
                    }
                } else {
                    const float *ap = A.a_int + fbase + (size_t)(E * t) * M + p;
                    float av[E];
#pragma unroll
                    for (int jj = 0; jj < E; ++jj) av[jj] = __ldcs(ap + (size_t)jj * M);
                    if constexpr (MODE == FRAME_ERR) {
                        const float fm = (float)M, inv_m = 1.0f / (float)M;
                        float sa = 0.f;
#pragma unroll
                        for (int jj = 0; jj < E; ++jj) {
                            const float mag2 = v[jj].x * v[jj].x + v[jj].y * v[jj].y;
                            const float a = av[jj] * fm;
                            if (mag2 > thr2) {
                                const float d = a - sqrtf(mag2) * inv_m;
                                sa += d * d;
                            } else {
                                const float dx = a - v[jj].x * inv_m, dy = v[jj].y * inv_m;
                                sa += dx * dx + dy * dy;
                            }
                        }
                        e_a += (double)sa;
                    } else {
#pragma unroll
                        for (int jj = 0; jj < E; ++jj) {
                            const float mag2 = v[jj].x * v[jj].x + v[jj].y * v[jj].y;
                            const float oa = om * av[jj];
                            if (mag2 > thr2) {
                                const float sc = fmaf(oa, rsqrtf(mag2), bm);
                                v[jj].x *= sc;
                                v[jj].y *= sc;
                            } else {
                                v[jj].x = fmaf(bm, v[jj].x, oa);
                                v[jj].y = bm * v[jj].y;
                            }
                        }
                        dft_b<E, RB, +1>(v);
#pragma unroll
                        for (int jj = 0; jj < E; jj += 2)
                            row4[((E * t + jj) ^ swzB) >> 1] = make_float4(v[jj].x, v[jj].y, v[jj + 1].x, v[jj + 1].y);
                    }
                }
            }
            __syncthreads();
            if constexpr (MODE == FRAME_ITER) {
                const float2 *row = strip + lineA * M;
#pragma unroll
                for (int k = 0; k < E; ++k) v[k] = row[(s + k * TPL) ^ swzA];
#pragma unroll
                for (int k = 1; k < E; ++k) v[k] = cmulc(v[k], tw.get(k));
                dft<E, +1>(v);
                float2 *dst = scr + (size_t)(p0 + lineA) * M;
#pragma unroll
                for (int j = 0; j < E; ++j) st_l2(dst + s + j * TPL, v[j]);
            }
        }
        if (CS > 1) cluster_barrier(); else __syncthreads();

        // ---------------- stage 3: rows.  load transposed, B^-1, exchange, A^-1, store c --------------------
        if constexpr (MODE == FRAME_ITER) {
            for (int sp = crank; sp < C::NSTRIP; sp += CS) {
                const int r0 = sp * L;
                float2 v[E];
                {
                    const float2 *src = scr + (size_t)(E * t) * M + (r0 + lineB);
#pragma unroll
                    for (int jj = 0; jj < E; ++jj) v[jj] = ld_l2(src + (size_t)jj * M);
                    dft_b<E, RB, +1>(v);
                    float4 *row4 = reinterpret_cast<float4 *>(strip + lineB * M);
#pragma unroll
                    for (int jj = 0; jj < E; jj += 2)
                        row4[((E * t + jj) ^ swzB) >> 1] = make_float4(v[jj].x, v[jj].y, v[jj + 1].x, v[jj + 1].y);
                }
                __syncthreads();
                {
                    const float2 *row = strip + lineA * M;
#pragma unroll
                    for (int k = 0; k < E; ++k) v[k] = row[(s + k * TPL) ^ swzA];
#pragma unroll
                    for (int k = 1; k < E; ++k) v[k] = cmulc(v[k], tw.get(k));
                    dft<E, +1>(v);
                    float2 *dst = A.c_out + fbase + (size_t)(r0 + lineA) * M;
#pragma unroll
                    for (int j = 0; j < E; ++j) st_stream(dst + s + j * TPL, v[j]);
                }
                __syncthreads();
            }
            if (CS > 1) cluster_barrier();   // the next frame's stage 1 overwrites the scratch the others still read
        }
    }

    if constexpr (MODE == FRAME_ERR) {
        // deterministic block reduction of the three sums (fixed tree), one triple per CTA
        __syncthreads();
        double *red = reinterpret_cast<double *>(smem_raw);
        red[tid] = e_a;
        red[NT + tid] = e_q;
        red[2 * NT + tid] = e_d;
        __syncthreads();
        for (int off = NT / 2; off > 0; off >>= 1) {
            if (tid < off) {
                red[tid] += red[tid + off];
                red[NT + tid] += red[NT + tid + off];
                red[2 * NT + tid] += red[2 * NT + tid + off];
            }
            __syncthreads();
        }
        if (tid == 0) {
            A.err_partials[3 * blockIdx.x + 0] = red[0];
            A.err_partials[3 * blockIdx.x + 1] = red[NT];
            A.err_partials[3 * blockIdx.x + 2] = red[2 * NT];
        }
    }
}

}  // namespace sharp
