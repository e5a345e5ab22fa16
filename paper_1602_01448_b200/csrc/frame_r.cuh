// frame_r.cuh -- the fused per-frame kernel for frames that fit one SM (m = 64, 128): steps a1-a4 and the
// frame-local half of a6.  What one frame goes through (Eq. 7,
// :174-178 step 5):
//     z  = c_prev + w_form . T_i psi_v
//     Z^ = FFT2_unnormalised(z)                             (= m F z, F the unitary DFT of Eq. 2)
//     C^ = Z^ (beta/m^2 + (1-2 beta)(a/m)/|Z^|)             (|F z| > thr; else C^ = beta/m^2 Z^ + (1-2 beta) a/m: G4)
//     c  = IFFT2_unnormalised(C^) = beta z + (1 - 2 beta) P_a z
//
// Radix plan ("5 + 5 + LB x LB"): every thread holds 32 complex values in registers, the CTA has m^2/32 threads, so
// one sweep of a pass covers the whole frame and a frame makes exactly five register passes with four exchanges
// through shared memory between them (8 shared-memory accesses per pixel in all, nothing else is staged):
//
//   P1   global -> registers.  Thread = (column c = 32 cblk + lane, r_lo); registers i: rows r = r_lo + NLO i.
//        Lanes run along a row of the frame: every load / store instruction of a warp is one contiguous 256-byte
//        segment.  z is formed on the fly (probe from tensor memory at m = 128).  DFT32 over i -> u1.
//   X1   CTA-wide exchange (barrier 1).
//   P2   thread = (warp = u1 >> SPB, lane = (c_lo, r_lo, u1_low)); registers j: columns c = c_lo + NLO j.
//        DFT32 over j -> v1.
//   X2   exchange inside the warp (padded 32 x 34 transposition, __syncwarp only).
//   P3   thread = (same warp, lane = v1); registers q = (u1_low, r_lo, c_lo).  Twiddles W^{u1 r_lo}, W^{v1 c_lo},
//        DFT_NLO over r_lo -> u2 and over c_lo -> v2: Z^(u1 + 32 u2, v1 + 32 v2).  Projection.  Then the same
//        steps backwards with conjugated twiddles: P3^-1, X2^-1, P2^-1, X1^-1 (barrier 2), P1^-1 -> global.
//
// LB = log2(m) - 5 (1, 2), NLO = 2^LB, SPB = 5 - 2 LB "spare" register bits in P3 (u1_low).  Two CTA barriers per
// frame: a thread re-writes in X1 of the next frame exactly the locations it read in X1^-1, and the warp-private
// exchanges X2 live in the region of the exchange buffer that only this warp reads in X1.
//
// Exchange buffer: NW regions (one per P2 warp) of RS = 1152 slots of 8 bytes; all address functions are sums of a
// per-thread base and a compile-time function of the register index (immediate offsets, no swizzle arithmetic);
// the paddings (36, 144, 576 / 66, 132, 264, 528; row pitch 34) make every access bank-conflict free.
// The amplitudes are stored in the order P3 reads them: a_int[(warp 32 + q) 32 + lane] (see slot_freq()).
//
// Latency: the state and the amplitudes of the next frame are pulled into L2 by one bulk prefetch each, a whole
// frame ahead (measured: 262 us per launch at config 2 with it, 301 us without, and no better when issued later);
// the position of the next frame is fetched a frame ahead as well.  Variants measured and dropped (config 2, us per
// launch): amplitudes staged in shared memory by a bulk copy 298; object tile or amplitudes by cp.async into
// slots of the exchange buffer the thread owns at that time 265 / 302; object tile requested before the state 297.
#pragma once
#include "fft_regs.cuh"
#include "frame_common.cuh"

#ifndef SHARP_STAGGER_NS
#define SHARP_STAGGER_NS 1700
#endif
#ifndef SHARP_STAGGER_PHASES
#define SHARP_STAGGER_PHASES 8
#endif
#ifndef SHARP_DYN
#define SHARP_DYN 1
#endif
#ifndef SHARP_R_PIPE
#define SHARP_R_PIPE 1
#endif
#ifndef SHARP_R_EARLY
#define SHARP_R_EARLY 0
#endif

namespace sharp {

template <int M>
struct RCfg {
    static_assert(M == 64 || M == 128, "register-radix frame kernel: m = 64 or 128");
    static constexpr int LB = (M == 128) ? 2 : 1;
    static constexpr int NLO = 1 << LB;
    static constexpr int SPB = 5 - 2 * LB, SP = 1 << SPB;
    static constexpr int NT = M * M / 32, NW = NT / 32, CB = M / 32;
    static constexpr int RS = 1152;                       // slots per region
    static constexpr int XE = (M == 128) ? 36 : 66;       // X1 pitch of r_lo
    static constexpr int X2P = 34;                        // X2 row pitch
    static constexpr int E_BYTES = NW * RS * 8;
    static constexpr int TW_BYTES = M * 8;
    static constexpr int SMEM_BYTES = E_BYTES + TW_BYTES + 64;
    static constexpr bool W_TMEM = (M == 128);            // probe parked in tensor memory
    static constexpr int MIN_CTAS = (M == 128) ? 1 : 3;
    SHARP_HD static constexpr int xc(int c) { return M == 128 ? (c & 31) + 144 * (c >> 5) : c; }
    SHARP_HD static constexpr int xu(int u)
    {
        return M == 128 ? 576 * u : 132 * (u & 1) + 264 * ((u >> 1) & 1) + 528 * (u >> 2);
    }
    // X1 offset of register j in P2 (column c = c_lo + NLO j) relative to the thread's base
    SHARP_HD static constexpr int x1j(int j) { return M == 128 ? 4 * (j & 7) + 144 * (j >> 3) : 2 * j; }
    // X1 offset of register u1 in P1
    SHARP_HD static constexpr int x1u(int u1) { return (u1 >> SPB) * RS + xu(u1 & (SP - 1)); }
};

// Amplitude slot -> frequency: slot = (warp 32 + q) 32 + lane holds a(u, v), u = (warp SP + u1_low) + 32 u2,
// v = lane + 32 v2, q = v2 + NLO u2 + NLO^2 u1_low: a warp's load of register q is 128 contiguous bytes.
template <int M>
SHARP_HD void slot_freq(int slot, int &u, int &v)
{
    using C = RCfg<M>;
    const int lane = slot & 31, q = (slot >> 5) & 31, warp = slot >> 10;
    const int v2 = q & (C::NLO - 1), u2 = (q >> C::LB) & (C::NLO - 1), u1_low = q >> (2 * C::LB);
    u = warp * C::SP + u1_low + 32 * u2;
    v = lane + 32 * v2;
}

// ---- the passes, as functions of (thread id, exchange buffer): the kernel below and the host emulation used by
// ---- the unit tests of the index algebra run exactly this code -------------------------------------------------
template <int M>
struct RPass {
    using C = RCfg<M>;

    // X1 write in the P1 mapping (and X1^-1 read)
    SHARP_HD static int p1_base(int tid)
    {
        const int wq = tid >> 5, lane = tid & 31;
        const int r_lo = wq % C::NLO, cblk = wq / C::NLO;
        return C::xc(32 * cblk + lane) + C::XE * r_lo;
    }
    SHARP_HD static void p1_store(int tid, float2 *E, const float2 *v)
    {
        float2 *b = E + p1_base(tid);
#pragma unroll
        for (int u1 = 0; u1 < 32; ++u1) b[C::x1u(u1)] = v[u1];
    }
    SHARP_HD static void p1_load(int tid, const float2 *E, float2 *v)
    {
        const float2 *b = E + p1_base(tid);
#pragma unroll
        for (int u1 = 0; u1 < 32; ++u1) v[u1] = b[C::x1u(u1)];
    }
    // X1 read in the P2 mapping (and X1^-1 write)
    SHARP_HD static int p2_base(int tid)
    {
        const int wq = tid >> 5, lane = tid & 31;
        const int c_lo = lane & (C::NLO - 1), r_lo = (lane >> C::LB) & (C::NLO - 1), u1_low = lane >> (2 * C::LB);
        return wq * C::RS + C::xu(u1_low) + C::XE * r_lo + c_lo;
    }
    SHARP_HD static void p2_load(int tid, const float2 *E, float2 *v)
    {
        const float2 *b = E + p2_base(tid);
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = b[C::x1j(j)];
    }
    SHARP_HD static void p2_store(int tid, float2 *E, const float2 *v)
    {
        float2 *b = E + p2_base(tid);
#pragma unroll
        for (int j = 0; j < 32; ++j) b[C::x1j(j)] = v[j];
    }
    // X2: register v1 of lane q  <->  register q of lane v1
    SHARP_HD static void x2_store_cols(int tid, float2 *E, const float2 *v)
    {
        float2 *b = E + (tid >> 5) * C::RS + (tid & 31);
#pragma unroll
        for (int v1 = 0; v1 < 32; ++v1) b[C::X2P * v1] = v[v1];
    }
    SHARP_HD static void x2_load_cols(int tid, const float2 *E, float2 *v)
    {
        const float2 *b = E + (tid >> 5) * C::RS + (tid & 31);
#pragma unroll
        for (int v1 = 0; v1 < 32; ++v1) v[v1] = b[C::X2P * v1];
    }
    SHARP_HD static void x2_load_rows(int tid, const float2 *E, float2 *v)
    {
        const float4 *b = reinterpret_cast<const float4 *>(E + (tid >> 5) * C::RS + C::X2P * (tid & 31));
#pragma unroll
        for (int q = 0; q < 32; q += 2) {
            const float4 t = b[q >> 1];
            v[q] = make_float2(t.x, t.y);
            v[q + 1] = make_float2(t.z, t.w);
        }
    }
    SHARP_HD static void x2_store_rows(int tid, float2 *E, const float2 *v)
    {
        float4 *b = reinterpret_cast<float4 *>(E + (tid >> 5) * C::RS + C::X2P * (tid & 31));
#pragma unroll
        for (int q = 0; q < 32; q += 2) b[q >> 1] = make_float4(v[q].x, v[q].y, v[q + 1].x, v[q + 1].y);
    }

    // P3 forward: twiddles + DFT_NLO over r_lo and c_lo for each u1_low; v[q] -> Z^ at q = v2 + NLO u2 + NLO^2 u1_low.
    // tw = table of W_M^k (k < M); t2[c_lo] = W_M^{v1 c_lo} (per-thread registers, c_lo >= 1).
    template <int SGN>
    SHARP_HD static void p3_small_dfts(float2 *v)
    {
#pragma unroll
        for (int s = 0; s < C::SP; ++s) {
            float2 *p = v + C::NLO * C::NLO * s;
            if (SGN < 0) {   // columns direction (over r_lo, stride NLO) first, then rows (over c_lo, stride 1)
#pragma unroll
                for (int cl = 0; cl < C::NLO; ++cl) Dft<C::NLO, SGN, C::NLO>::run(p + cl);
#pragma unroll
                for (int rl = 0; rl < C::NLO; ++rl) Dft<C::NLO, SGN, 1>::run(p + C::NLO * rl);
            } else {
#pragma unroll
                for (int rl = 0; rl < C::NLO; ++rl) Dft<C::NLO, SGN, 1>::run(p + C::NLO * rl);
#pragma unroll
                for (int cl = 0; cl < C::NLO; ++cl) Dft<C::NLO, SGN, C::NLO>::run(p + cl);
            }
        }
    }
    // multiplies v[(s, r_lo, c_lo)] by W^{+-(u1 r_lo)} W^{+-(v1 c_lo)}; CONJ selects the inverse
    template <bool CONJ>
    SHARP_HD static void p3_twiddle(int tid, const float2 *tw, const float2 *t2, float2 *v)
    {
        const int wq = tid >> 5;
#pragma unroll
        for (int s = 0; s < C::SP; ++s) {
            const int u1 = wq * C::SP + s;
#pragma unroll
            for (int rl = 0; rl < C::NLO; ++rl) {
                float2 t1 = make_float2(1.f, 0.f);
                if (rl > 0) t1 = tw[(u1 * rl) & (M - 1)];
#pragma unroll
                for (int cl = 0; cl < C::NLO; ++cl) {
                    float2 &x = v[cl + C::NLO * rl + C::NLO * C::NLO * s];
                    if (CONJ) {
                        if (cl > 0) x = cmulc(x, t2[cl]);
                        if (rl > 0) x = cmulc(x, t1);
                    } else {
                        if (rl > 0) x = cmul(x, t1);
                        if (cl > 0) x = cmul(x, t2[cl]);
                    }
                }
            }
        }
    }
};

// The forward twiddle is applied BEFORE the small DFTs, the inverse one AFTER the small inverse DFTs.

#if defined(__CUDACC__)

// WRAP: the object index r + x_i is taken modulo the image size (periodic boundary of the Fig. 3 simulation, reading G25);
// a separate instantiation, so the plain kernel pays nothing for it.
template <int M, int MODE, bool WRAP = false>
__global__ void __launch_bounds__(RCfg<M>::NT, RCfg<M>::MIN_CTAS) k_frame_r(FrameArgs A)
{
    using C = RCfg<M>;
    using P = RPass<M>;
    constexpr int NLO = C::NLO, NT = C::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *E = reinterpret_cast<float2 *>(smem_raw);
    float2 *tw = reinterpret_cast<float2 *>(smem_raw + C::E_BYTES);
    unsigned *tmem_slot = reinterpret_cast<unsigned *>(smem_raw + C::E_BYTES + C::TW_BYTES);

    const int tid = threadIdx.x, wq = tid >> 5, lane = tid & 31;
    // P1 identity
    const int r_lo = wq % NLO, cblk = wq / NLO, col = 32 * cblk + lane;

    // FRAME_ITER pipelines the state loads with the previous frame's stores: register v[k] is re-loaded with the next
    // frame's value right after it has been stored (the loads enter the LSU queue between the stores instead of behind all
    // of them), so the frame's own load of c happens only before a CTA's first frame.  Measured: 242.7 -> 241.2 us at
    // config 2, 937 -> 900 us per 10,000 frames at config 6.  Issuing that first load before the twiddle / tensor-memory
    // set-up and the start-up stagger (SHARP_R_EARLY) is slower, 244.3 against 241.4 us: all SMs then load in step again.
    constexpr bool PIPE = (MODE == FRAME_ITER) && (SHARP_R_PIPE != 0);
    float2 v[32];
    if (PIPE && SHARP_R_EARLY && (int)blockIdx.x < A.K) {
        const float2 *cin = A.c_in + (size_t)blockIdx.x * M * M + (size_t)r_lo * M + col;
#pragma unroll
        for (int k = 0; k < 32; ++k) v[k] = ld_stream(cin + (size_t)k * (NLO * M));
    }

    for (int k = tid; k < M; k += NT) {
        float sn, cs;
        sincospif(-2.0f * (float)k / (float)M, &sn, &cs);
        tw[k] = make_float2(cs, sn);
    }
    // P3 identity: lane = v1; row twiddles W^{v1 c_lo}
    float2 t2[NLO];
#pragma unroll
    for (int cl = 0; cl < NLO; ++cl) {
        float sn, cs;
        sincospif(-2.0f * (float)((lane * cl) & (M - 1)) / (float)M, &sn, &cs);
        t2[cl] = make_float2(cs, sn);
    }

    // probe -> tensor memory, once per launch: this thread's 32 probe values (rows r_lo + NLO i of column col) sit in
    // its own TMEM lane, columns 64 cblk .. 64 cblk + 63
    const bool use_w = (MODE != FRAME_FFT) && A.psi_v != nullptr;
    const bool w_tmem = C::W_TMEM && MODE == FRAME_ITER && use_w;
    unsigned tw_addr = 0;
    if (w_tmem) {
        if (wq == 0) r_tmem_alloc(tmem_slot, 256);
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        tw_addr = *reinterpret_cast<volatile unsigned *>(tmem_slot) + ((unsigned)(32 * (wq & 3)) << 16) + 64u * (unsigned)cblk;
#pragma unroll 1
        for (int ch = 0; ch < 4; ++ch) {
            float2 wv[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) wv[k] = __ldg(A.w_form + (r_lo + NLO * (8 * ch + k)) * M + col);
            r_tmem_st16(tw_addr + 16 * ch, wv);
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    } else {
        __syncthreads();
    }

    const float thr2 = A.sc->thr2;
    const float bm = A.bm, om = A.om;
    double s_a = 0.0, s_q = 0.0, s_d = 0.0;

    // Frame schedule.  What a CTA needs to know about its next frame (index, position) is CTA-uniform, so it lives in a
    // double-buffered shared-memory slot instead of registers: thread 0 fills slot (n+1)&1 during frame n (before barrier
    // 1) and everybody reads it at the top of frame n+1.  The first frame of a CTA is its own index; with SHARP_DYN every
    // further one comes from a global counter (integer atomicAdd: a CTA that is ahead takes more frames), otherwise it
    // is the fixed round-robin.  FRAME_ERR always uses the round-robin: its per-CTA partial sums must group the same
    // frames on every run (bitwise reproducible residuals).
    constexpr bool DYN = (MODE != FRAME_ERR) && (SHARP_DYN != 0);
    volatile int *s_sched = reinterpret_cast<volatile int *>(smem_raw + C::E_BYTES + C::TW_BYTES + 16);   // [2][4]
    if (blockIdx.x == 0 && tid == 0) *A.sched_next = 0;          // the next launch's counter (launches are stream-ordered)

#if SHARP_STAGGER_NS > 0
    // All CTAs start together, so for the first rounds every SM loads, computes and stores at the same time and the
    // HBM bursts (47 MB per round at m = 128) are not hidden behind anybody's butterflies: measured 17.3 us per round
    // in lockstep against 13.5 us once the SMs have drifted apart.  Start the CTAs in SHARP_STAGGER_PHASES phases
    // instead.  Measured at config 2 (us per launch, dynamic schedule): no stagger 262; 2 x 6800 ns 242.1; 3 x 4500 242.1;
    // 4 x 3400 243.6; 4 x 4000 245.6; 6 x 2300 242.4; 8 x 1700 242.2; 8 x 2200 245.2.  With the fixed round-robin: 261 / 250.
    if (MODE == FRAME_ITER && A.K > 2 * (int)gridDim.x) {
        const unsigned delay = (blockIdx.x % (unsigned)SHARP_STAGGER_PHASES) * (unsigned)SHARP_STAGGER_NS;
        unsigned long long t0, t1;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
        do { asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1)); } while (t1 - t0 < delay);
    }
#endif

    if (tid == 0) {
        const int i0 = blockIdx.x;
        s_sched[0] = i0;
        if (i0 < A.K) {
            s_sched[1] = __ldg(A.pos + 2 * i0);
            s_sched[2] = __ldg(A.pos + 2 * i0 + 1);
            prefetch_l2_bulk(A.c_in + (size_t)i0 * M * M, M * M * 8);
            if (MODE != FRAME_FFT) prefetch_l2_bulk(A.a_int + (size_t)i0 * M * M, M * M * 4);
        }
    }
    __syncthreads();

    if (PIPE && !SHARP_R_EARLY) {
        const int i0 = s_sched[0];
        if (i0 < A.K) {
            const float2 *cin = A.c_in + (size_t)i0 * M * M + (size_t)r_lo * M + col;
#pragma unroll
            for (int k = 0; k < 32; ++k) v[k] = ld_stream(cin + (size_t)k * (NLO * M));
        }
    }

    for (int par = 0;; par ^= 1) {
        const int i = s_sched[4 * par];
        if (i >= A.K) break;
        const int xr = s_sched[4 * par + 1], xc = s_sched[4 * par + 2];
        const size_t fbase = (size_t)i * M * M;
        // thread 0 asks for the next frame now and consumes the answers just before barrier 1, when this frame's own
        // loads have long been issued
        int i_next = i + (int)gridDim.x, ticket = 0, nxr = 0, nxc = 0;
        if (tid == 0) {
            if (DYN) {
                ticket = atomicAdd(A.sched, 1);
            } else if (i_next < A.K) {
                nxr = __ldg(A.pos + 2 * i_next);
                nxc = __ldg(A.pos + 2 * i_next + 1);
                prefetch_l2_bulk(A.c_in + (size_t)i_next * M * M, M * M * 8);
                if (MODE != FRAME_FFT) prefetch_l2_bulk(A.a_int + (size_t)i_next * M * M, M * M * 4);
            }
        }

        // ---------------- P1: form z, DFT32 down the column -----------------------------------------------
        {
            if (!PIPE) {
                const float2 *cin = A.c_in + fbase + (size_t)r_lo * M + col;
#pragma unroll
                for (int k = 0; k < 32; ++k) v[k] = ld_stream(cin + (size_t)k * (NLO * M));
            }
            if (MODE == FRAME_FFT && A.conj_io) {
#pragma unroll
                for (int k = 0; k < 32; ++k) v[k].y = -v[k].y;
            }
            if (use_w) {
                const float2 *prow = A.psi_v + (size_t)(xr + r_lo) * A.nc + xc + col;
                const size_t pstep = (size_t)NLO * A.nc;
                int pcw = xc + col;                  // WRAP only
                if (WRAP && pcw >= A.nc) pcw -= A.nc;
#pragma unroll
                for (int ch = 0; ch < 4; ++ch) {
                    float2 pv[8], wv[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        if constexpr (WRAP) {
                            int prw = xr + r_lo + NLO * (8 * ch + k);
                            if (prw >= A.nr) prw -= A.nr;
                            pv[k] = __ldg(A.psi_v + (size_t)prw * A.nc + pcw);
                        } else {
                            pv[k] = __ldg(prow + (size_t)(8 * ch + k) * pstep);
                        }
                    }
                    if (w_tmem) {
                        r_tmem_ld16(tw_addr + 16 * ch, wv);
                    } else {
#pragma unroll
                        for (int k = 0; k < 8; ++k) wv[k] = __ldg(A.w_form + (r_lo + NLO * (8 * ch + k)) * M + col);
                    }
#pragma unroll
                    for (int k = 0; k < 8; ++k) v[8 * ch + k] = cadd(v[8 * ch + k], cmul(wv[k], pv[k]));
                }
            }
            if constexpr (MODE == FRAME_ERR) {
                float sq, sd;
                frame_err_qd32<M, NLO>(A, v, fbase, xr, xc, r_lo, col, sq, sd);
                s_q += (double)sq;
                s_d += (double)sd;
            }
            dft<32, -1>(v);
            P::p1_store(tid, E, v);
        }
        if (tid == 0) {
            if (DYN) {
                i_next = (int)gridDim.x + ticket;
                if (i_next < A.K) {
                    nxr = __ldg(A.pos + 2 * i_next);
                    nxc = __ldg(A.pos + 2 * i_next + 1);
                    prefetch_l2_bulk(A.c_in + (size_t)i_next * M * M, M * M * 8);
                    if (MODE != FRAME_FFT) prefetch_l2_bulk(A.a_int + (size_t)i_next * M * M, M * M * 4);
                }
            }
            s_sched[4 * (par ^ 1)] = i_next;
            s_sched[4 * (par ^ 1) + 1] = nxr;
            s_sched[4 * (par ^ 1) + 2] = nxc;
        }
        __syncthreads();                                                     // barrier 1
        const int i_follow = PIPE ? s_sched[4 * (par ^ 1)] : 0;             // the frame after this one (uniform)
        // ---------------- P2: DFT32 along the row ----------------------------------------------------------
        P::p2_load(tid, E, v);
        dft<32, -1>(v);
        __syncwarp();
        P::x2_store_cols(tid, E, v);
        __syncwarp();
        // ---------------- P3: last radix-NLO stages, projection, and back ----------------------------------
        P::x2_load_rows(tid, E, v);
        P::template p3_twiddle<false>(tid, tw, t2, v);
        P::template p3_small_dfts<-1>(v);
        if constexpr (MODE == FRAME_FFT) {
            const float inv_m = 1.0f / (float)M;
#pragma unroll
            for (int q = 0; q < 32; ++q) {
                int u, vv;
                slot_freq<M>((wq * 32 + q) * 32 + lane, u, vv);
                float2 o = make_float2(v[q].x * inv_m, v[q].y * inv_m);
                if (A.conj_io) o.y = -o.y;
                A.c_out[fbase + (size_t)u * M + vv] = o;
            }
            __syncthreads();     // X1 of the next frame re-uses the regions the other warps still read
            continue;
        } else {
            const float *ap = A.a_int + fbase + (size_t)(wq * 32) * 32 + lane;
            if constexpr (MODE == FRAME_ERR) {
                s_a += (double)frame_err_a32<M>(v, ap, thr2);
                __syncthreads();
                continue;
            } else {
#pragma unroll
                for (int q0 = 0; q0 < 32; q0 += 8) {
                    float av[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) av[k] = __ldcs(ap + (q0 + k) * 32);
                    frame_project8(v + q0, av, thr2, bm, om);
                }
            }
        }
        if constexpr (MODE == FRAME_ITER) {
            P::template p3_small_dfts<+1>(v);
            P::template p3_twiddle<true>(tid, tw, t2, v);
            P::x2_store_rows(tid, E, v);
            __syncwarp();
            // ---------------- P2^-1 ------------------------------------------------------------------------
            P::x2_load_cols(tid, E, v);
            dft<32, +1>(v);
            __syncwarp();
            P::p2_store(tid, E, v);
            __syncthreads();                                                 // barrier 2
            // ---------------- P1^-1 -> global --------------------------------------------------------------
            P::p1_load(tid, E, v);
            dft<32, +1>(v);
            float2 *dst = A.c_out + fbase + (size_t)r_lo * M + col;
            if (PIPE && i_follow < A.K) {
                const float2 *cin = A.c_in + (size_t)i_follow * M * M + (size_t)r_lo * M + col;
#pragma unroll
                for (int k = 0; k < 32; ++k) {
                    st_stream(dst + (size_t)k * (NLO * M), v[k]);
                    v[k] = ld_stream(cin + (size_t)k * (NLO * M));
                }
            } else {
#pragma unroll
                for (int k = 0; k < 32; ++k) st_stream(dst + (size_t)k * (NLO * M), v[k]);
            }
        }
    }
    if (w_tmem) {
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (wq == 0) r_tmem_dealloc(*reinterpret_cast<volatile unsigned *>(tmem_slot), 256);
    }

    if constexpr (MODE == FRAME_ERR) frame_err_reduce(s_a, s_q, s_d, smem_raw, C::NW, A.err_partials);
}

#endif  // __CUDACC__

}  // namespace sharp
