// frame_ws.cuh -- the iteration kernel for m = 128, warp-specialised.
//
// Same arithmetic, pass structure and shared-memory frame layout as frame_smem.cuh (steps a1-a4 + the frame half
// of a6: z = c + w . T psi_v, FFT2, magnitude projection folded with the RAAR frame combine, IFFT2).  What is new
// is who touches global memory:
//
//   * one PRODUCER warpgroup (4 warps, 64 registers/thread) forms z = c + w_form . T psi_v for the rows of the
//     NEXT frame with fully coalesced 128-bit loads and writes them into a ring of six 16-row slots in shared
//     memory (96 KB), signalling one mbarrier per slot.  It runs up to 96 rows ahead of the consumers, i.e. it
//     works while they are in the column stage and the inverse row stage of the current frame, so none of the
//     state / probe / object load latency is on the FFT warps' critical path;
//   * four CONSUMER warpgroups (16 warps, 104 registers/thread, `setmaxnreg`) run the eight radix passes on the
//     frame buffer F (128 KB).  They are split in two groups of 256 threads that own the row strips
//     [64 g, 64 g + 64) in the row stages and the column strips with the same numbers in the column stage; passes
//     inside a stage synchronise with a per-group named barrier only, the three stage changes with a
//     consumer-wide one.
//
// Ring protocol: the eight 16-row chunks q of a frame are produced in the order j(q) the two groups consume them
// (q = 0,1,4,5,2,3,6,7); chunk number n = 8 * frame_seq + j lives in slot n % 6; full[slot] (128 producer arrivals)
// completes its (n / 6)-th phase when the chunk is written; empty[slot] (4 consumer-warp arrivals) completes it
// when the four warps that read the chunk hold it in registers.
#pragma once
#include "frame_smem.cuh"

namespace sharp {

struct WsCfg {
    static constexpr int M = 128, E = 16, TPL = 8, RB = 8, RA = 16;
    static constexpr int NCONS = 512, NPROD = 128, NT = NCONS + NPROD, GSZ = 256, L = 32;  // L: lines per group pass
    static constexpr int SR = 16, NSLOT = 6, CHUNKS = M / SR;                                // ring geometry
    static constexpr int F_BYTES = M * M * 8, S_BYTES = NSLOT * SR * M * 8;
    static constexpr int SMEM_BYTES = F_BYTES + S_BYTES + 2 * NSLOT * 8;
    // setmaxnreg moves registers inside the CTA's own pool (640 threads x 96 at launch = 61440), so the two
    // budgets must satisfy 512 * REGS_CONS + 128 * REGS_PROD <= 61440 or the increase blocks for ever.
    static constexpr int REGS_LAUNCH = 96, REGS_CONS = 104, REGS_PROD = 64;
    static_assert(NCONS * REGS_CONS + NPROD * REGS_PROD <= NT * REGS_LAUNCH, "setmaxnreg budgets exceed the CTA pool");
};

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(void *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void *bar)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(void *bar, unsigned parity)
{
    unsigned ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(void *bar, unsigned parity)
{
    // a protocol error must surface as a launch failure (SHARP_ECUDA), never as a hung GPU
    for (unsigned spins = 0; !mbar_try_wait(bar, parity); ++spins)
        if (spins > (1u << 26)) __trap();
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
template <int N>
__device__ __forceinline__ void reg_dec()
{
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N));
}
template <int N>
__device__ __forceinline__ void reg_inc()
{
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N));
}

// production order of the eight 16-row chunks of a frame: position j -> chunk q, and its inverse
__device__ __forceinline__ int ws_chunk_of(int j) { return (j & 1) | ((j & 2) << 1) | ((j & 4) >> 1); }
__device__ __forceinline__ int ws_seq_of(int q) { return (q & 1) | ((q & 4) >> 1) | ((q & 2) << 1); }

__global__ void __launch_bounds__(WsCfg::NT, 1) k_frame_ws128(FrameArgs A)
{
    using C = WsCfg;
    constexpr int M = C::M, E = C::E, TPL = C::TPL, RB = C::RB, L = C::L, SR = C::SR, NSLOT = C::NSLOT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *F = reinterpret_cast<float2 *>(smem_raw);
    float2 *S = reinterpret_cast<float2 *>(smem_raw + C::F_BYTES);
    unsigned long long *full = reinterpret_cast<unsigned long long *>(smem_raw + C::F_BYTES + C::S_BYTES);
    unsigned long long *empty = full + NSLOT;

    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int k = 0; k < NSLOT; ++k) {
            mbar_init(full + k, C::NPROD);
            mbar_init(empty + k, 4);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid >= C::NCONS) {
        // =========================== producer warpgroup ==================================================
        reg_dec<C::REGS_PROD>();
        const int pw = (tid - C::NCONS) >> 5, lane = tid & 31;
        if (pw == 0 && lane == 0 && (int)blockIdx.x < A.K) {
            prefetch_l2_bulk(A.c_in + (size_t)blockIdx.x * M * M, M * M * 8);
            prefetch_l2_bulk(A.a_int + (size_t)blockIdx.x * M * M, M * M * 4);
        }
        int n = 0;  // chunk counter of this CTA
        for (int i = blockIdx.x; i < A.K; i += gridDim.x) {
            const int xr = A.pos[2 * i], xc = A.pos[2 * i + 1];
            const size_t fbase = (size_t)i * M * M;
            if (pw == 0 && lane == 0 && i + (int)gridDim.x < A.K) {
                const size_t nb = (size_t)(i + gridDim.x) * M * M;
                prefetch_l2_bulk(A.c_in + nb, M * M * 8);
                prefetch_l2_bulk(A.a_int + nb, M * M * 4);
            }
#pragma unroll 1
            for (int j = 0; j < C::CHUNKS; ++j, ++n) {
                const int slot = n % NSLOT, fill = n / NSLOT;
                if (fill > 0) mbar_wait(empty + slot, (unsigned)((fill - 1) & 1));
                const int q = ws_chunk_of(j);
                float2 *Sslot = S + slot * (SR * M);
#pragma unroll
                for (int half = 0; half < 2; ++half) {
                    // this warp's rows 4 pw + 2 half + {0, 1} of the chunk; lane: pixels 2 lane, 2 lane + 1 and +64
                    float4 cv[2][2], wv[2][2];
                    float2 pv[2][4];
#pragma unroll
                    for (int rr = 0; rr < 2; ++rr) {
                        const int rl = 4 * pw + 2 * half + rr, r = q * SR + rl;
                        const float4 *c4 = reinterpret_cast<const float4 *>(A.c_in + fbase + (size_t)r * M);
                        cv[rr][0] = __ldcs(c4 + lane);
                        cv[rr][1] = __ldcs(c4 + 32 + lane);
                    }
                    if (A.psi_v != nullptr) {
#pragma unroll
                        for (int rr = 0; rr < 2; ++rr) {
                            const int rl = 4 * pw + 2 * half + rr, r = q * SR + rl;
                            const float4 *w4 = reinterpret_cast<const float4 *>(A.w_form + r * M);
                            wv[rr][0] = __ldg(w4 + lane);
                            wv[rr][1] = __ldg(w4 + 32 + lane);
                            const float2 *prow = A.psi_v + (size_t)(xr + r) * A.nc + xc;
                            pv[rr][0] = __ldg(prow + 2 * lane);
                            pv[rr][1] = __ldg(prow + 2 * lane + 1);
                            pv[rr][2] = __ldg(prow + 64 + 2 * lane);
                            pv[rr][3] = __ldg(prow + 64 + 2 * lane + 1);
                        }
#pragma unroll
                        for (int rr = 0; rr < 2; ++rr)
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                const float2 z0 = cadd(make_float2(cv[rr][h].x, cv[rr][h].y),
                                                       cmul(make_float2(wv[rr][h].x, wv[rr][h].y), pv[rr][2 * h]));
                                const float2 z1 = cadd(make_float2(cv[rr][h].z, cv[rr][h].w),
                                                       cmul(make_float2(wv[rr][h].z, wv[rr][h].w), pv[rr][2 * h + 1]));
                                cv[rr][h] = make_float4(z0.x, z0.y, z1.x, z1.y);
                            }
                    }
#pragma unroll
                    for (int rr = 0; rr < 2; ++rr) {
                        const int rl = 4 * pw + 2 * half + rr, r = q * SR + rl;
                        float4 *d4 = reinterpret_cast<float4 *>(Sslot + rl * M);
                        const int sw = swz_row(r);
                        d4[((2 * lane) ^ sw) >> 1] = cv[rr][0];
                        d4[((64 + 2 * lane) ^ sw) >> 1] = cv[rr][1];
                    }
                }
                mbar_arrive(full + slot);
            }
        }
        return;
    }

    // =============================== consumer warpgroups ===================================================
    reg_inc<C::REGS_CONS>();
    const int g = tid / C::GSZ, gtid = tid % C::GSZ;       // group, thread in group
    const int lineA = gtid / TPL, s = gtid % TPL;           // A / X mappings (32 lines, 8 threads each)
    const int lineB = gtid % L, t = gtid / L;               // B / Y mappings (32 lines, t in 0..7)
    const int warp_in_group = gtid >> 5, lane = tid & 31;
    const int bar_g = 1 + g;

    Twiddles<M, E> tw;
    tw.init(nullptr, s, tid, C::NCONS);
    const int swX = swz_row(s);                             // rows s + 8 j: (row & 7) == s

    const float thr2 = A.sc->thr2;
    const float bm = A.bm, om = A.om;

    int fseq = 0;
    for (int i = blockIdx.x; i < A.K; i += gridDim.x, ++fseq) {
        const size_t fbase = (size_t)i * M * M;

        if (g == 1 && A.stagger_ns > 0) __nanosleep(A.stagger_ns);
        // ---------------- stage 1: rows of this group.  staged z -> pass A -> exchange -> pass B ---------------
#pragma unroll 1
        for (int u = 0; u < 2; ++u) {
            const int r0 = 64 * g + 32 * u;
            float2 v[E];
            {
                const int r = r0 + lineA;
                const int q = 4 * g + 2 * u + (warp_in_group >> 2);   // lineA / 16
                const int n = fseq * C::CHUNKS + ws_seq_of(q);
                const int slot = n % NSLOT;
                mbar_wait(full + slot, (unsigned)((n / NSLOT) & 1));
                const float2 *src = S + slot * (SR * M) + (lineA & (SR - 1)) * M;
                const int sw = swz_row(r);
#pragma unroll
                for (int j = 0; j < E; ++j) v[j] = src[(s + j * TPL) ^ sw];
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + slot);
                dft<E, -1>(v);
#pragma unroll
                for (int k = 1; k < E; ++k) v[k] = cmul(v[k], tw.get(k));
                float2 *row = F + r * M;
#pragma unroll
                for (int k = 0; k < E; ++k) row[(s + k * TPL) ^ sw] = v[k];
            }
            named_bar_sync(bar_g, C::GSZ);
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
        named_bar_sync(3, C::NCONS);
        if (g == 1 && A.stagger_ns > 0) __nanosleep(A.stagger_ns);

        // ---------------- stage 2: columns of this group.  X, Y (project), X^-1 ----------------------------------
#pragma unroll 1
        for (int u = 0; u < 2; ++u) {
            const int p0 = 64 * g + 32 * u;
            float2 v[E];
            const int pX = (p0 + lineA) ^ swX;
            {
#pragma unroll
                for (int j = 0; j < E; ++j) v[j] = F[(s + j * TPL) * M + pX];
                dft<E, -1>(v);
#pragma unroll
                for (int k = 1; k < E; ++k) v[k] = cmul(v[k], tw.get(k));
#pragma unroll
                for (int k = 0; k < E; ++k) F[(s + k * TPL) * M + pX] = v[k];
            }
            named_bar_sync(bar_g, C::GSZ);
            {
                const int p = p0 + lineB;
                float av[E];
                const float *ap = A.a_int + fbase + (size_t)(E * t) * M + p;
#pragma unroll
                for (int jj = 0; jj < E; ++jj) av[jj] = __ldcs(ap + (size_t)jj * M);
#pragma unroll
                for (int jj = 0; jj < E; ++jj) v[jj] = F[(E * t + jj) * M + (p ^ swz_row(jj))];
                dft_b<E, RB, -1>(v);
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
            named_bar_sync(bar_g, C::GSZ);
            {
#pragma unroll
                for (int k = 0; k < E; ++k) v[k] = F[(s + k * TPL) * M + pX];
#pragma unroll
                for (int k = 1; k < E; ++k) v[k] = cmulc(v[k], tw.get(k));
                dft<E, +1>(v);
#pragma unroll
                for (int j = 0; j < E; ++j) F[(s + j * TPL) * M + pX] = v[j];
            }
        }
        named_bar_sync(3, C::NCONS);
        if (g == 1 && A.stagger_ns > 0) __nanosleep(A.stagger_ns);

        // ---------------- stage 3: rows of this group.  pass B^-1, exchange, pass A^-1, store c' -----------------
#pragma unroll 1
        for (int u = 0; u < 2; ++u) {
            const int r0 = 64 * g + 32 * u;
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
            named_bar_sync(bar_g, C::GSZ);
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
    }
}

}  // namespace sharp
