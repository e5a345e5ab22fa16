// frame_ws.cuh -- the iteration kernel for m = 128, warp-specialised.
//
// Same arithmetic, pass structure and shared-memory frame layout as frame_smem.cuh (steps a1-a4 + the frame half
// of a6: z = c + w . T psi_v, FFT2, magnitude projection folded with the RAAR frame combine, IFFT2).  What is new
// is who touches global memory:
//
//   * one PRODUCER warpgroup (4 warps) stages z = c + w_form . T psi_v for the rows of the NEXT frame: the state c
//     goes straight from global into the staging slot with cp.async (16-byte copies, no registers, all four rows
//     of a warp in flight), the object tile comes through registers with coalesced 64-bit loads, the probe is parked
//     once per launch in the producer threads' own TMEM lanes (128 KB of the SM's 256 KB tensor memory) and read
//     back with tcgen05.ld, so it costs L2 -> SM bandwidth once per launch instead of once per frame,
//     and each thread then combines in place the locations it copied itself.  Six 16-row chunks go to a ring in
//     shared memory (96 KB, one full/empty mbarrier pair per slot), the last two (rows 96..127) in place into the
//     frame buffer once the consumers have retired those rows, so a whole frame is staged ahead and none of the
//     state / probe / object load latency is on the FFT warps' critical path;
//   * four CONSUMER warpgroups (16 warps) run the eight radix passes on the frame buffer F (128 KB).  They are
//     split in two groups of 256 threads that own the row strips [64 g, 64 g + 64) in the row stages and the
//     column strips with the same numbers in the column stage; passes inside a stage synchronise with a per-group
//     named barrier only, the three stage changes with a consumer-wide one.  Group 1 runs its strips in the
//     order (1, 0) in the inverse row stage so that rows 96..127 retire early.
//   All 640 threads run at the launch budget of 96 registers (an earlier variant moved registers from the
//   producer to the consumers with setmaxnreg; the pool of 640 x 96 left the consumers only 104, which bought
//   nothing).
//
// Ring protocol: chunk q of 16 rows has sequence number j(q) in the order the two groups consume them
// (q = 0,1,4,5,2,3,6,7).  j < 6: slot j of the ring; full[j] (128 producer arrivals) completes its phase
// `frame_seq` when the chunk is written, empty[j] (4 consumer-warp arrivals) when the four warps that read it hold
// it in registers.  j = 6, 7: fullF[j - 6] likewise; emptyF (8 warp arrivals) completes when group 1 has read rows
// 96..127 of the previous frame for the last time.
#pragma once
#include "frame_smem.cuh"

namespace sharp {

struct WsCfg {
    static constexpr int M = 128, E = 16, TPL = 8, RB = 8, RA = 16;
    static constexpr int NCONS = 512, NPROD = 128, NT = NCONS + NPROD, GSZ = 256, L = 32;  // L: lines per group pass
    static constexpr int SR = 16, NSLOT = 6, CHUNKS = M / SR;                                // ring geometry
    static constexpr int F_BYTES = M * M * 8, S_BYTES = NSLOT * SR * M * 8;
    static constexpr int SMEM_BYTES = F_BYTES + S_BYTES + (2 * NSLOT + 3) * 8 + 8;   // + TMEM base slot
    static constexpr int REGS_LAUNCH = 96;   // 640 threads x 96 registers = 61440 of the SM's 65536
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
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity), "r"(0x989680u)   // suspend-time hint (ns)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(void *bar, unsigned parity)
{
    // a protocol error must surface as a launch failure (SHARP_ECUDA), never as a hung GPU
    for (unsigned spins = 0; !mbar_try_wait(bar, parity); ++spins)
        if (spins > (1u << 22)) __trap();
}
__device__ __forceinline__ void cp_async_16(void *smem_dst, const void *gmem_src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void named_bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
// Tensor memory (TMEM, 256 KB per SM, otherwise idle in this kernel) as a register-file extension of the producer:
// a thread's probe values are the same for every frame, so they are parked once per launch in the thread's own
// TMEM lane (32 rows x 4 pixels x 8 bytes = 256 columns) and read back with tcgen05.ld when a chunk is combined.
__device__ __forceinline__ void tmem_alloc_256(unsigned *smem_slot)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" ::"r"(smem_u32(smem_slot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_256(unsigned taddr)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" ::"r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st8(unsigned taddr, const float4 &a, const float4 &b)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr),
                 "r"(__float_as_uint(a.x)), "r"(__float_as_uint(a.y)), "r"(__float_as_uint(a.z)), "r"(__float_as_uint(a.w)),
                 "r"(__float_as_uint(b.x)), "r"(__float_as_uint(b.y)), "r"(__float_as_uint(b.z)), "r"(__float_as_uint(b.w))
                 : "memory");
}
__device__ __forceinline__ void tmem_ld8(unsigned taddr, float4 &a, float4 &b)
{
    unsigned r0, r1, r2, r3, r4, r5, r6, r7;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3), "=r"(r4), "=r"(r5), "=r"(r6), "=r"(r7)
                 : "r"(taddr)
                 : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    a = make_float4(__uint_as_float(r0), __uint_as_float(r1), __uint_as_float(r2), __uint_as_float(r3));
    b = make_float4(__uint_as_float(r4), __uint_as_float(r5), __uint_as_float(r6), __uint_as_float(r7));
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
    unsigned long long *fullF = empty + NSLOT;   // [2]: chunks 6, 7 are produced in place in F rows 96..127
    unsigned long long *emptyF = fullF + 2;      // group 1 has retired F rows 96..127 (8 warp arrivals)
    unsigned *tmem_slot = reinterpret_cast<unsigned *>(emptyF + 1);

    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int k = 0; k < NSLOT; ++k) {
            mbar_init(full + k, C::NPROD);
            mbar_init(empty + k, 4);
        }
        mbar_init(fullF + 0, C::NPROD);
        mbar_init(fullF + 1, C::NPROD);
        mbar_init(emptyF, 8);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid >= C::NCONS) {
        // =========================== producer warpgroup ==================================================
        const int pw = (tid - C::NCONS) >> 5, lane = tid & 31;
        if (pw == 0 && lane == 0 && (int)blockIdx.x < A.K) {
            prefetch_l2_bulk(A.c_in + (size_t)blockIdx.x * M * M, M * M * 8);
            prefetch_l2_bulk(A.a_int + (size_t)blockIdx.x * M * M, M * M * 4);
        }
        // probe -> TMEM, once per launch (lanes 32 pw .. 32 pw + 31 belong to this warp)
        const bool w_tmem = A.psi_v != nullptr;
        unsigned tw_addr = 0;
        if (w_tmem) {
            if (pw == 0) tmem_alloc_256(tmem_slot);
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            named_bar_sync(4, C::NPROD);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            tw_addr = *reinterpret_cast<volatile unsigned *>(tmem_slot) + ((unsigned)(32 * pw) << 16);
#pragma unroll 1
            for (int qr = 0; qr < 32; ++qr) {   // qr = 4 q + rr
                const int r = (qr >> 2) * SR + 4 * pw + (qr & 3);
                const float4 *w4 = reinterpret_cast<const float4 *>(A.w_form + r * M);
                tmem_st8(tw_addr + 8 * qr, __ldg(w4 + lane), __ldg(w4 + 32 + lane));
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        }
        int fseq = 0;  // frames this CTA has staged
        for (int i = blockIdx.x; i < A.K; i += gridDim.x, ++fseq) {
            const int xr = A.pos[2 * i], xc = A.pos[2 * i + 1];
            const size_t fbase = (size_t)i * M * M;
            if (pw == 0 && lane == 0 && i + (int)gridDim.x < A.K) {
                const size_t nb = (size_t)(i + gridDim.x) * M * M;
                prefetch_l2_bulk(A.c_in + nb, M * M * 8);
                prefetch_l2_bulk(A.a_int + nb, M * M * 4);
            }
#pragma unroll 1
            for (int j = 0; j < C::CHUNKS; ++j) {
                // chunks j = 0..5 go to ring slot j; j = 6, 7 (rows 96..127) in place into F once group 1 has
                // retired those rows of the previous frame (it runs that strip first in stage 3)
                const bool inF = j >= NSLOT;
                if (fseq > 0) mbar_wait(inF ? emptyF : empty + j, (unsigned)((fseq - 1) & 1));
                const int q = ws_chunk_of(j);
                float2 *Sslot = inF ? F + q * (SR * M) : S + j * (SR * M);
                // this warp's rows 4 pw + {0..3} of the chunk; lane: pixels 2 lane, 2 lane + 1 and the same + 64.
                // The state c goes straight into the slot with cp.async (no registers: all four rows in flight),
                // the probe and the object tile through registers; each thread then combines in place the
                // locations it copied itself, so no barrier is needed before the arrive.
#pragma unroll
                for (int rr = 0; rr < 4; ++rr) {
                    const int rl = 4 * pw + rr, r = q * SR + rl;
                    const float2 *crow = A.c_in + fbase + (size_t)r * M;
                    float2 *drow = Sslot + rl * M;
                    const int sw = swz_row(r);
                    cp_async_16(drow + ((2 * lane) ^ sw), crow + 2 * lane);
                    cp_async_16(drow + ((64 + 2 * lane) ^ sw), crow + 64 + 2 * lane);
                }
                cp_async_commit();
                if (A.psi_v != nullptr) {
                    float4 wv[4][2];
                    float2 pv[4][4];
#pragma unroll
                    for (int rr = 0; rr < 4; ++rr) {
                        const int r = q * SR + 4 * pw + rr;
                        const float2 *prow = A.psi_v + (size_t)(xr + r) * A.nc + xc;
                        pv[rr][0] = __ldg(prow + 2 * lane);
                        pv[rr][1] = __ldg(prow + 2 * lane + 1);
                        pv[rr][2] = __ldg(prow + 64 + 2 * lane);
                        pv[rr][3] = __ldg(prow + 64 + 2 * lane + 1);
                    }
#pragma unroll
                    for (int rr = 0; rr < 4; ++rr) tmem_ld8(tw_addr + 8 * (4 * q + rr), wv[rr][0], wv[rr][1]);
                    cp_async_wait_all();
#pragma unroll
                    for (int rr = 0; rr < 4; ++rr) {
                        const int rl = 4 * pw + rr, r = q * SR + rl;
                        float4 *d4 = reinterpret_cast<float4 *>(Sslot + rl * M);
                        const int sw = swz_row(r);
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            float4 *slot4 = d4 + (((64 * h + 2 * lane) ^ sw) >> 1);
                            const float4 cv = *slot4;
                            const float2 z0 = cadd(make_float2(cv.x, cv.y),
                                                   cmul(make_float2(wv[rr][h].x, wv[rr][h].y), pv[rr][2 * h]));
                            const float2 z1 = cadd(make_float2(cv.z, cv.w),
                                                   cmul(make_float2(wv[rr][h].z, wv[rr][h].w), pv[rr][2 * h + 1]));
                            *slot4 = make_float4(z0.x, z0.y, z1.x, z1.y);
                        }
                    }
                } else {
                    cp_async_wait_all();
                }
                mbar_arrive(inF ? fullF + (j - NSLOT) : full + j);
            }
        }
        if (w_tmem) {
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            named_bar_sync(4, C::NPROD);
            if (pw == 0) tmem_dealloc_256(*reinterpret_cast<volatile unsigned *>(tmem_slot));
        }
        return;
    }

    // =============================== consumer warpgroups ===================================================
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

        // ---------------- stage 1: rows of this group.  staged z -> pass A -> exchange -> pass B ---------------
#pragma unroll 1
        for (int u = 0; u < 2; ++u) {
            const int r0 = 64 * g + 32 * u;
            float2 v[E];
            {
                const int r = r0 + lineA;
                const int q = 4 * g + 2 * u + (warp_in_group >> 2);   // lineA / 16
                const int j = ws_seq_of(q);
                const int sw = swz_row(r);
                if (j < NSLOT) {
                    mbar_wait(full + j, (unsigned)(fseq & 1));
                    const float2 *src = S + j * (SR * M) + (lineA & (SR - 1)) * M;
#pragma unroll
                    for (int jj = 0; jj < E; ++jj) v[jj] = src[(s + jj * TPL) ^ sw];
                    __syncwarp();
                    if (lane == 0) mbar_arrive(empty + j);
                } else {   // rows 96..127: staged in place; the eight threads of a row sit in this warp
                    mbar_wait(fullF + (j - NSLOT), (unsigned)(fseq & 1));
                    const float2 *src = F + r * M;
#pragma unroll
                    for (int jj = 0; jj < E; ++jj) v[jj] = src[(s + jj * TPL) ^ sw];
                    __syncwarp();
                }
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

        // ---------------- stage 3: rows of this group.  pass B^-1, exchange, pass A^-1, store c' -----------------
#pragma unroll 1
        for (int uu = 0; uu < 2; ++uu) {
            const int u = uu ^ g;                           // group 1 retires rows 96..127 first (producer refills them)
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
                if (g == 1 && uu == 0) {
                    __syncwarp();
                    if (lane == 0) mbar_arrive(emptyF);
                }
#pragma unroll
                for (int k = 1; k < E; ++k) v[k] = cmulc(v[k], tw.get(k));
                dft<E, +1>(v);
                float2 *dst = A.c_out + fbase + (size_t)r * M;
#pragma unroll
                for (int j = 0; j < E; ++j) st_stream(dst + s + j * TPL, v[j]);
            }
        }
        // group 1 ends stage 3 on the strip it starts the next frame's stage 1 with: its readers must be done
        if (g == 1) named_bar_sync(bar_g, C::GSZ);
    }
}

}  // namespace sharp
