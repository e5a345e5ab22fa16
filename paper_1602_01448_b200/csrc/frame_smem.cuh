// frame_smem.cuh -- the fused per-frame kernel for frames that fit one SM's shared memory (m = 64, 128):
// form z, 2-D FFT, Fourier-magnitude projection folded with the frame-local half of RAAR, inverse 2-D FFT
// (steps a1-a4 + frame half of a6).  Same arithmetic and the same index algebra as
// frame_kernel.cuh (see its header for the DIF/DIT pass structure and the "position space" of the Fourier data);
// what differs is where the frame lives between the passes: the whole m x m frame stays in shared memory (128 KB
// at m = 128), so a frame-iteration touches HBM exactly once for the state read (8 B/px), once for the amplitudes
// (4 B/px) and once for the state write (8 B/px), and nothing round-trips through L2 between F and F*.
//
// Shared layout: element (row, pos) at row * M + (pos ^ swz(row)), swz(row) = bitrev3(row & 7) << 1 -- conflict
// free for all six access patterns below (64-bit and 128-bit).
//
// Thread mappings (E = 16 elements per thread, TPL = M/16 threads per line, L = 16 NT / M lines per strip):
//   rows,    A: thread (row = r0 + tid / TPL, s = tid % TPL) holds positions s + j TPL      (coalesced global rows)
//   rows,    B: thread (row = r0 + tid % L,   t = tid / L)   holds positions 16 t .. 16 t+15 (128-bit shared)
//   columns, X: thread (col = p0 + tid / TPL, s = tid % TPL) holds rows s + j TPL            (same twiddles as A)
//   columns, Y: thread (col = p0 + tid % L,   t = tid / L)   holds rows 16 t .. 16 t+15      (coalesced amplitudes)
//
// The next frame of this CTA (state and amplitudes) is prefetched into L2 with one bulk-prefetch instruction each
// while the current frame is being transformed, so the loads of stage 1 and of the projection are L2 hits.
#pragma once
#include "frame_kernel.cuh"

namespace sharp {

template <int M, int NT>
struct SmemFrameCfg {
    static constexpr int E = 16, RA = 16, RB = M / 16, TPL = M / 16, L = E * NT / M, NSTRIP = M / L;
    static constexpr int SMEM_BYTES = M * M * 8;
    static_assert(M % 16 == 0 && (E * NT) % M == 0 && M % L == 0 && L % 32 == 0, "bad frame configuration");
};

__device__ __forceinline__ int swz_row(int row) { return (int)((__brev((unsigned)(row & 7)) >> 29) << 1); }

__device__ __forceinline__ void prefetch_l2_bulk(const void *p, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

template <int M, int NT, int MODE>
__global__ void __launch_bounds__(NT, (NT <= 256 ? 2 : 1)) k_frame_smem(FrameArgs A)
{
    using C = SmemFrameCfg<M, NT>;
    constexpr int E = C::E, TPL = C::TPL, L = C::L, RB = C::RB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *F = reinterpret_cast<float2 *>(smem_raw);

    const int tid = threadIdx.x;
    const int lineA = tid / TPL, s = tid % TPL;
    const int lineB = tid % L, t = tid / L;

    Twiddles<M, E> tw;
    tw.init(nullptr, s, tid, NT);
    // X mapping: rows q = s + j TPL, so q & 7 takes one value (TPL = 8) or two (TPL = 4, by the parity of j)
    const int swX0 = swz_row(s), swX1 = swz_row(s + TPL);
    auto swX = [&](int j) { return ((j * TPL) & 7) ? swX1 : swX0; };

    const float thr2 = A.sc->thr2;
    const float bm = A.bm, om = A.om;
    double e_a = 0.0, e_q = 0.0, e_d = 0.0;

    if (tid == 0 && (int)blockIdx.x < A.K) {
        prefetch_l2_bulk(A.c_in + (size_t)blockIdx.x * M * M, M * M * 8);
        if (MODE != FRAME_FFT) prefetch_l2_bulk(A.a_int + (size_t)blockIdx.x * M * M, M * M * 4);
    }

    for (int i = blockIdx.x; i < A.K; i += gridDim.x) {
        const int xr = A.pos[2 * i], xc = A.pos[2 * i + 1];
        const size_t fbase = (size_t)i * M * M;
        if (tid == 0 && i + (int)gridDim.x < A.K) {
            const size_t nb = (size_t)(i + gridDim.x) * M * M;
            prefetch_l2_bulk(A.c_in + nb, M * M * 8);
            if (MODE != FRAME_FFT) prefetch_l2_bulk(A.a_int + nb, M * M * 4);
        }

        // ---------------- stage 1: rows.  form z, pass A, exchange, pass B (in place) ----------------------
#pragma unroll 1
        for (int sp = 0; sp < C::NSTRIP; ++sp) {
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
                float2 *row = F + r * M;
                const int sw = swz_row(r);
#pragma unroll
                for (int k = 0; k < E; ++k) row[(s + k * TPL) ^ sw] = v[k];
            }
            __syncthreads();
            {
                const int r = r0 + lineB;
                float4 *row4 = reinterpret_cast<float4 *>(F + r * M);
                const int sw = swz_row(r);
#pragma unroll
                for (int jj = 0; jj < E; jj += 2) {
                    float4 q4 = row4[((E * t + jj) ^ sw) >> 1];
                    v[jj] = make_float2(q4.x, q4.y);
                    v[jj + 1] = make_float2(q4.z, q4.w);
                }
                dft_b<E, RB, -1>(v);
#pragma unroll
                for (int jj = 0; jj < E; jj += 2)
                    row4[((E * t + jj) ^ sw) >> 1] = make_float4(v[jj].x, v[jj].y, v[jj + 1].x, v[jj + 1].y);
            }
        }
        __syncthreads();

        // ---------------- stage 2: columns.  X (pass A), Y (pass B, project, pass B^-1), X (pass A^-1) -------
#pragma unroll 1
        for (int sp = 0; sp < C::NSTRIP; ++sp) {
            const int p0 = sp * L;
            float2 v[E];
            const int pX = p0 + lineA;
            {
#pragma unroll
                for (int j = 0; j < E; ++j) {
                    const int q = s + j * TPL;
                    v[j] = F[q * M + (pX ^ swX(j))];
                }
                dft<E, -1>(v);
#pragma unroll
                for (int k = 1; k < E; ++k) v[k] = cmul(v[k], tw.get(k));
#pragma unroll
                for (int k = 0; k < E; ++k) {
                    const int q = s + k * TPL;
                    F[q * M + (pX ^ swX(k))] = v[k];
                }
            }
            __syncthreads();
            {
                const int p = p0 + lineB;
                float av[E];
                if constexpr (MODE != FRAME_FFT) {
                    const float *ap = A.a_int + fbase + (size_t)(E * t) * M + p;
#pragma unroll
                    for (int jj = 0; jj < E; ++jj) av[jj] = __ldcs(ap + (size_t)jj * M);
                }
#pragma unroll
                for (int jj = 0; jj < E; ++jj) v[jj] = F[(E * t + jj) * M + (p ^ swz_row(jj))];
                dft_b<E, RB, -1>(v);
                // v[jj] = Z^ at (q = E t + jj, p) in position space
                if constexpr (MODE == FRAME_FFT) {
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
                } else if constexpr (MODE == FRAME_ERR) {
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
                    for (int jj = 0; jj < E; ++jj) F[(E * t + jj) * M + (p ^ swz_row(jj))] = v[jj];
                }
            }
            if constexpr (MODE == FRAME_ITER) {
                __syncthreads();
#pragma unroll
                for (int k = 0; k < E; ++k) {
                    const int q = s + k * TPL;
                    v[k] = F[q * M + (pX ^ swX(k))];
                }
#pragma unroll
                for (int k = 1; k < E; ++k) v[k] = cmulc(v[k], tw.get(k));
                dft<E, +1>(v);
#pragma unroll
                for (int j = 0; j < E; ++j) {
                    const int q = s + j * TPL;
                    F[q * M + (pX ^ swX(j))] = v[j];
                }
            }
        }
        __syncthreads();

        // ---------------- stage 3: rows.  pass B^-1, exchange, pass A^-1, store c ----------------------------
        if constexpr (MODE == FRAME_ITER) {
#pragma unroll 1
            for (int sp = 0; sp < C::NSTRIP; ++sp) {
                const int r0 = sp * L;
                float2 v[E];
                {
                    const int r = r0 + lineB;
                    float4 *row4 = reinterpret_cast<float4 *>(F + r * M);
                    const int sw = swz_row(r);
#pragma unroll
                    for (int jj = 0; jj < E; jj += 2) {
                        float4 q4 = row4[((E * t + jj) ^ sw) >> 1];
                        v[jj] = make_float2(q4.x, q4.y);
                        v[jj + 1] = make_float2(q4.z, q4.w);
                    }
                    dft_b<E, RB, +1>(v);
#pragma unroll
                    for (int jj = 0; jj < E; jj += 2)
                        row4[((E * t + jj) ^ sw) >> 1] = make_float4(v[jj].x, v[jj].y, v[jj + 1].x, v[jj + 1].y);
                }
                __syncthreads();
                {
                    const int r = r0 + lineA;
                    const float2 *row = F + r * M;
                    const int sw = swz_row(r);
#pragma unroll
                    for (int k = 0; k < E; ++k) v[k] = row[(s + k * TPL) ^ sw];
#pragma unroll
                    for (int k = 1; k < E; ++k) v[k] = cmulc(v[k], tw.get(k));
                    dft<E, +1>(v);
                    float2 *dst = A.c_out + fbase + (size_t)r * M;
#pragma unroll
                    for (int j = 0; j < E; ++j) st_stream(dst + s + j * TPL, v[j]);
                }
            }
            if (C::NSTRIP == 1) __syncthreads();   // the next frame's stage 1 overwrites the rows just read
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
