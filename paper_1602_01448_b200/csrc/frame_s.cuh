// frame_s.cuh -- the fused per-frame kernel for frames larger than one SM's shared memory (m = 256, 512): steps
// a1-a4 and the frame-local half of a6 (same arithmetic as frame_r.cuh, see its header).
//
// A frame is processed in STRIPS of 8192 values (256 threads x 32 registers; 74 KB of shared memory, so two CTAs
// with independent phases share an SM) by the CS CTAs of a thread-block cluster.  m = 32 NLO (NLO = 8, 16).
//
//   stage 1, column strips (WC = 8192/m columns each; CTA q takes strips q, q + CS, ...):
//     P1  global -> registers, lanes along a row (coalesced 256 / 128 byte runs), registers i: rows r_lo + NLO i;
//         z = c + w T psi_v formed on the fly; DFT32 over i -> u1.
//     X1  CTA-wide exchange in shared memory (padded, bank-conflict free, immediate offsets).
//     P2  registers (r_lo, sp): twiddle W_m^{u1 r_lo}, DFT_NLO over r_lo -> u2 (u = u1 + 32 u2); the result goes to
//         the cluster's scratch frame in L2 in the order stage 2 reads it.
//   -- cluster barrier --
//   stage 2, row strips (WC rows each):
//     P3  scratch -> registers (coalesced: thread = (c_lo, u_lo) x warp, registers j: columns c_lo + NLO j);
//         DFT32 over j -> v1.
//     X3  32 x 32 transposition inside the warp (pitch 34).
//     P4  twiddle W_m^{v1 c_lo}, DFT_NLO over c_lo -> v2 (v = v1 + 32 v2); magnitude projection against the
//         amplitudes (stored in exactly this order); the same steps backwards; scratch written in place.
//   -- cluster barrier --
//   stage 3, column strips: P2^-1 (scratch -> registers, same addresses the thread wrote in stage 1), X1^-1, P1^-1
//     -> global.  Stage 1 of the cluster's next frame follows without a barrier (a thread only re-writes scratch
//     locations it has just read itself).
//
// Measured at config-4 size (1,600 frames, us per launch): 256-thread CTAs in clusters of 4: 1098; 128-thread CTAs
// (m = 256: strips of 16 columns, four CTAs per SM) in clusters of 8: 929, in clusters of 4: 1212; the probe parked in
// tensor memory (4 x 128 columns per SM): 1821 (the allocations of the four resident CTAs serialise), dropped.  Clusters
// started in phases (what helps frame_r.cuh): 863 without, 863 / 869 with 8 phases of 2.5 / 5 us: no effect, dropped.
// Resident CTAs per SM at m = 256 (128 threads; registers per thread): 3 (168) 916 us, 4 (128, small spill) 814 us, 5 (96) 1051 us,
// 6 (80) 1378 us; at m = 512 (256 threads) 2 (128) 4.66 ms, 3 (80) 8.60 ms.
// A per-line L2 prefetch of the CTA's next stage-1 strips, issued between the arrive and the wait of the second cluster
// barrier (one stage ahead only): 861 against 863 at m = 256, 5.12 against 4.97 ms at config 5: dropped.
// A bulk L2 prefetch of the cluster's next frame (what frame_r.cuh does) costs here: 926 with, 865 without (config 5:
// 5.45 / 4.99 ms): the prefetched frames push the scratch frames out of L2.
// The scratch frame (m^2 c64 per cluster) is the only data that leaves the SM between F and F*; it is re-used for
// every frame of the cluster and stays in L2 (evict-last policy; state / amplitudes stream with evict-first).
// Scratch element (u, c): index ((u >> SPB) 32 + (c >> LB)) 32 + ((u & (SP-1)) << LB) + (c & (NLO-1)).
#pragma once
#include "fft_regs.cuh"
#include "frame_common.cuh"

#ifndef SHARP_S_MINB
#define SHARP_S_MINB(nt) (512 / (nt))
#endif
#ifndef SHARP_S_PIPE
#define SHARP_S_PIPE 1
#endif

namespace sharp {

template <int M, int NT_>
struct SCfg {
    static_assert((M == 256 && (NT_ == 256 || NT_ == 128)) || (M == 512 && NT_ == 256), "strip frame kernel: m = 256 or 512");
    static constexpr int LB = (M == 256) ? 3 : 4, NLO = 1 << LB;
    static constexpr int SPB = 5 - LB, SP = 1 << SPB;
    static constexpr int NT = NT_, NW = NT / 32;
    static constexpr int WC = NT * 32 / M, NSTR = M / WC;     // strip width (columns / rows), strips per stage
    static constexpr int UW = WC >> SPB;                      // P3 warps (blocks of SP rows) per row strip == NW
    static constexpr int RS = 1088, X2P = 34;
    static constexpr int E_BYTES = NW * RS * 8, TW_BYTES = M * 8;
    static constexpr int SMEM_BYTES = E_BYTES + TW_BYTES + 64;
    static constexpr bool HALF = (NT == 128);                 // m = 256 in strips of 16 columns
    static_assert(UW == NW, "row strips: one P3 warp per SP rows");
    // X1 offsets of register u1 (P1 side) and of register rho = r_lo + NLO sp (P2 side); region = P2 warp
    SHARP_HD static constexpr int x1u(int u1)
    {
        return HALF ? ((u1 >> 2) & 3) * RS + 136 * (u1 & 3) + 544 * (u1 >> 4)
             : M == 256 ? (u1 >> 2) * RS + 264 * (u1 & 3)
                        : ((u1 >> 1) & 7) * RS + 256 * (u1 & 1) + 512 * (u1 >> 4);
    }
    SHARP_HD static constexpr int x1r(int rho)
    {
        return HALF ? 16 * (rho & 7) + 8 * ((rho >> 3) & 1) + 544 * (rho >> 4)
             : M == 256 ? 32 * (rho & 7) + 8 * (rho >> 3)
                        : 16 * (rho & 15) + 512 * (rho >> 4);
    }
    SHARP_HD static constexpr int x1lane(int u1_lo) { return (HALF ? 136 : M == 256 ? 264 : 256) * u1_lo; }
};

// amplitude slot -> frequency (stage 2 order): slot = ((s2 8 + w3) 32 + q) 32 + lane, q = v2 + NLO u_lo
template <int M>
SHARP_HD void slot_freq_s(int slot, int &u, int &v)
{
    using C = SCfg<M, 256>;
    const int lane = slot & 31, q = (slot >> 5) & 31, uhi = slot >> 10;
    u = (uhi << C::SPB) + (q >> C::LB);
    v = lane + 32 * (q & (C::NLO - 1));
}

template <int M, int NT_>
struct SPass {
    using C = SCfg<M, NT_>;
    // ---- X1 -------------------------------------------------------------------------------------------------
    SHARP_HD static int p1_base(int tid) { return (tid % C::WC) + C::WC * (tid / C::WC); }
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
    SHARP_HD static int p2_base(int tid)
    {
        const int w2 = tid >> 5, lane = tid & 31;
        const int c_lo = lane & (C::NLO - 1), u1_lo = lane >> C::LB;
        return w2 * C::RS + c_lo + C::x1lane(u1_lo);
    }
    SHARP_HD static void p2_load(int tid, const float2 *E, float2 *v)
    {
        const float2 *b = E + p2_base(tid);
#pragma unroll
        for (int rho = 0; rho < 32; ++rho) v[rho] = b[C::x1r(rho)];
    }
    SHARP_HD static void p2_store(int tid, float2 *E, const float2 *v)
    {
        float2 *b = E + p2_base(tid);
#pragma unroll
        for (int rho = 0; rho < 32; ++rho) b[C::x1r(rho)] = v[rho];
    }
    // u1 of a P2 thread for spare index sp
    SHARP_HD static int p2_u1(int tid, int sp)
    {
        const int w2 = tid >> 5, u1_lo = (tid & 31) >> C::LB;
        return C::HALF ? 16 * (sp >> 1) + 4 * w2 + u1_lo : M == 256 ? 4 * w2 + u1_lo : 16 * sp + 2 * w2 + u1_lo;
    }
    // scratch index of register rho = u2 + NLO sp of a P2 thread working on column strip s1
    SHARP_HD static int p2_scratch(int tid, int s1, int rho)
    {
        const int w2 = tid >> 5, lane = tid & 31;
        const int u2 = rho & (C::NLO - 1), sp = rho >> C::LB;
        const int uhi = C::HALF ? 4 * (sp >> 1) + w2 + 8 * u2 : M == 256 ? w2 + 8 * u2 : 8 * sp + w2 + 16 * u2;
        const int j = C::HALF ? 2 * s1 + (sp & 1) : M == 256 ? 4 * s1 + sp : s1;
        return (uhi * 32 + j) * 32 + lane;
    }
    // twiddle + DFT_NLO over r_lo (forward) / inverse DFT_NLO + conjugate twiddle
    template <bool INV>
    SHARP_HD static void p2_math(int tid, const float2 *tw, float2 *v)
    {
#pragma unroll
        for (int sp = 0; sp < C::SP; ++sp) {
            float2 *p = v + C::NLO * sp;
            const int u1 = p2_u1(tid, sp);
            if (INV) Dft<C::NLO, +1, 1>::run(p);
#pragma unroll
            for (int rl = 1; rl < C::NLO; ++rl) {
                const float2 t = tw[(u1 * rl) & (M - 1)];
                p[rl] = INV ? cmulc(p[rl], t) : cmul(p[rl], t);
            }
            if (!INV) Dft<C::NLO, -1, 1>::run(p);
        }
    }
    // ---- stage 2 ----------------------------------------------------------------------------------------------
    SHARP_HD static int p3_scratch(int tid, int s2, int j) { return ((s2 * C::NW + (tid >> 5)) * 32 + j) * 32 + (tid & 31); }
    SHARP_HD static void x3_store_cols(int tid, float2 *E, const float2 *v)
    {
        float2 *b = E + (tid >> 5) * C::RS + (tid & 31);
#pragma unroll
        for (int v1 = 0; v1 < 32; ++v1) b[C::X2P * v1] = v[v1];
    }
    SHARP_HD static void x3_load_cols(int tid, const float2 *E, float2 *v)
    {
        const float2 *b = E + (tid >> 5) * C::RS + (tid & 31);
#pragma unroll
        for (int v1 = 0; v1 < 32; ++v1) v[v1] = b[C::X2P * v1];
    }
    SHARP_HD static void x3_load_rows(int tid, const float2 *E, float2 *v)
    {
        const float4 *b = reinterpret_cast<const float4 *>(E + (tid >> 5) * C::RS + C::X2P * (tid & 31));
#pragma unroll
        for (int q = 0; q < 32; q += 2) {
            const float4 t = b[q >> 1];
            v[q] = make_float2(t.x, t.y);
            v[q + 1] = make_float2(t.z, t.w);
        }
    }
    SHARP_HD static void x3_store_rows(int tid, float2 *E, const float2 *v)
    {
        float4 *b = reinterpret_cast<float4 *>(E + (tid >> 5) * C::RS + C::X2P * (tid & 31));
#pragma unroll
        for (int q = 0; q < 32; q += 2) b[q >> 1] = make_float4(v[q].x, v[q].y, v[q + 1].x, v[q + 1].y);
    }
    template <bool INV>
    SHARP_HD static void p4_math(int tid, const float2 *tw, float2 *v)
    {
        const int v1 = tid & 31;
        if (INV) {
#pragma unroll
            for (int ul = 0; ul < C::SP; ++ul) Dft<C::NLO, +1, 1>::run(v + C::NLO * ul);
        }
#pragma unroll
        for (int cl = 1; cl < C::NLO; ++cl) {
            const float2 t = tw[(v1 * cl) & (M - 1)];
#pragma unroll
            for (int ul = 0; ul < C::SP; ++ul) {
                float2 &x = v[cl + C::NLO * ul];
                x = INV ? cmulc(x, t) : cmul(x, t);
            }
        }
        if (!INV) {
#pragma unroll
            for (int ul = 0; ul < C::SP; ++ul) Dft<C::NLO, -1, 1>::run(v + C::NLO * ul);
        }
    }
};

#if defined(__CUDACC__)

__device__ __forceinline__ unsigned long long s_policy_evict_last()
{
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ float2 s_ld_scratch(const float2 *p, unsigned long long pol)
{
    float2 v;
    asm volatile("ld.global.cg.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol) : "memory");
    return v;
}
__device__ __forceinline__ void s_st_scratch(float2 *p, float2 v, unsigned long long pol)
{
    asm volatile("st.global.cg.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(v.x), "f"(v.y), "l"(pol) : "memory");
}

// Launched with cluster dimension CS; gridDim.x is a multiple of CS.  scratch: one m x m frame per cluster.
// WRAP: periodic object index (see frame_r.cuh).
template <int M, int NT_, int MODE, int CS, bool WRAP = false>
__global__ void __launch_bounds__(NT_, SHARP_S_MINB(NT_)) k_frame_s(FrameArgs A)
{
    using C = SCfg<M, NT_>;
    using P = SPass<M, NT_>;
    constexpr int NLO = C::NLO, NT = C::NT, WC = C::WC;
    static_assert(C::NSTR % CS == 0, "strips must divide evenly over the cluster");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *E = reinterpret_cast<float2 *>(smem_raw);
    float2 *tw = reinterpret_cast<float2 *>(smem_raw + C::E_BYTES);

    const int tid = threadIdx.x, wq = tid >> 5, lane = tid & 31;
    const int col_l = tid % WC, r_lo = tid / WC;        // P1 identity
    for (int k = tid; k < M; k += NT) {
        float sn, cs;
        sincospif(-2.0f * (float)k / (float)M, &sn, &cs);
        tw[k] = make_float2(cs, sn);
    }
    __syncthreads();

    const int crank = (int)cluster_rank();
    const int cid = blockIdx.x / CS, nclusters = gridDim.x / CS;
    float2 *scr = A.scratch + (size_t)cid * M * M;
    const unsigned long long pol_keep = s_policy_evict_last();
    const bool use_w = (MODE != FRAME_FFT) && A.psi_v != nullptr;
    const float thr2 = A.sc->thr2;
    const float bm = A.bm, om = A.om;
    double s_a = 0.0, s_q = 0.0, s_d = 0.0;

    // FRAME_ITER pipelines, at every strip transition, the loads of the next strip with the stores of the current one: register
    // v[k] is re-loaded right after it has been stored, so the loads enter the LSU queue between the stores instead of behind
    // all of them (stage 1: scratch stores / next strip's state; stage 2: scratch stores / next strip's scratch loads; stage 3:
    // global stores / next strip's scratch loads, and for the last strip the first stage-1 strip of the cluster's next frame).
    // Measured (us per launch at 1,600 frames of 256 x 256 / ms at config 5): none 866 / 4.95; frame transition only 840 / 4.92;
    // all transitions 814 / 4.66.
    constexpr bool PIPE = (MODE == FRAME_ITER) && (SHARP_S_PIPE != 0);
    bool preloaded = false;
    float2 v[32];
    for (int i = cid; i < A.K; i += nclusters) {
        const int xr = __ldg(A.pos + 2 * i), xc = __ldg(A.pos + 2 * i + 1);
        const size_t fbase = (size_t)i * M * M;

        // ---------------- stage 1: column strips ------------------------------------------------------------
        for (int s1 = crank; s1 < C::NSTR; s1 += CS) {
            const int col = s1 * WC + col_l;
            {
                if (!(PIPE && preloaded)) {
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
                    const float2 *wrow = A.w_form + (size_t)r_lo * M + col;
                    const size_t pstep = (size_t)NLO * A.nc;
                    int pcw = xc + col;              // WRAP only
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
#pragma unroll
                        for (int k = 0; k < 8; ++k) wv[k] = __ldg(wrow + (size_t)(8 * ch + k) * (NLO * M));
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
            }
            __syncthreads();                 // the previous strip's X1 readers are done
            P::p1_store(tid, E, v);
            __syncthreads();
            P::p2_load(tid, E, v);
            P::template p2_math<false>(tid, tw, v);
            preloaded = false;
            if (PIPE && s1 + CS < C::NSTR) {     // the next strip's state is requested between this strip's scratch stores
                const float2 *cin = A.c_in + fbase + (size_t)r_lo * M + (s1 + CS) * WC + col_l;
#pragma unroll
                for (int rho = 0; rho < 32; ++rho) {
                    s_st_scratch(scr + P::p2_scratch(tid, s1, rho), v[rho], pol_keep);
                    v[rho] = ld_stream(cin + (size_t)rho * (NLO * M));
                }
                preloaded = true;
            } else {
#pragma unroll
                for (int rho = 0; rho < 32; ++rho) s_st_scratch(scr + P::p2_scratch(tid, s1, rho), v[rho], pol_keep);
            }
        }
        // this thread's 32 amplitudes of a row strip are requested well ahead of the projection: for the first strip
        // between the arrive and the wait of the cluster barrier, for the others before the forward transform
        float av_all[32];
        auto load_amplitudes = [&](int s2) {
            if (MODE == FRAME_ITER) {
                const float *ap0 = A.a_int + fbase + (size_t)((s2 * C::NW + wq) * 32) * 32 + lane;
#pragma unroll
                for (int q = 0; q < 32; ++q) av_all[q] = __ldcs(ap0 + q * 32);
            }
        };
        cluster_arrive();
        load_amplitudes(crank);
        cluster_wait();

        // ---------------- stage 2: row strips ---------------------------------------------------------------
        for (int s2 = crank; s2 < C::NSTR; s2 += CS) {
            if (!(PIPE && preloaded)) {
#pragma unroll
                for (int j = 0; j < 32; ++j) v[j] = s_ld_scratch(scr + P::p3_scratch(tid, s2, j), pol_keep);
            }
            preloaded = false;
            if (s2 != crank) load_amplitudes(s2);
            dft<32, -1>(v);
            __syncwarp();
            P::x3_store_cols(tid, E, v);
            __syncwarp();
            P::x3_load_rows(tid, E, v);
            P::template p4_math<false>(tid, tw, v);
            const int uhi = s2 * C::NW + wq;
            if constexpr (MODE == FRAME_FFT) {
                const float inv_m = 1.0f / (float)M;
#pragma unroll
                for (int q = 0; q < 32; ++q) {
                    int u, vv;
                    slot_freq_s<M>((uhi * 32 + q) * 32 + lane, u, vv);
                    float2 o = make_float2(v[q].x * inv_m, v[q].y * inv_m);
                    if (A.conj_io) o.y = -o.y;
                    A.c_out[fbase + (size_t)u * M + vv] = o;
                }
            } else {
                const float *ap = A.a_int + fbase + (size_t)(uhi * 32) * 32 + lane;
                if constexpr (MODE == FRAME_ERR) {
                    s_a += (double)frame_err_a32<M>(v, ap, thr2);
                } else {
#pragma unroll
                    for (int q0 = 0; q0 < 32; q0 += 8) frame_project8(v + q0, av_all + q0, thr2, bm, om);
                    P::template p4_math<true>(tid, tw, v);
                    P::x3_store_rows(tid, E, v);
                    __syncwarp();
                    P::x3_load_cols(tid, E, v);
                    dft<32, +1>(v);
                    if (PIPE && s2 + CS < C::NSTR) {
#pragma unroll
                        for (int j = 0; j < 32; ++j) {
                            s_st_scratch(scr + P::p3_scratch(tid, s2, j), v[j], pol_keep);
                            v[j] = s_ld_scratch(scr + P::p3_scratch(tid, s2 + CS, j), pol_keep);
                        }
                        preloaded = true;
                    } else {
#pragma unroll
                        for (int j = 0; j < 32; ++j) s_st_scratch(scr + P::p3_scratch(tid, s2, j), v[j], pol_keep);
                    }
                }
            }
            __syncwarp();
        }
        cluster_arrive();
        cluster_wait();

        // ---------------- stage 3: column strips ------------------------------------------------------------
        if constexpr (MODE == FRAME_ITER) {
            for (int s1 = crank; s1 < C::NSTR; s1 += CS) {
                if (!(PIPE && preloaded)) {
#pragma unroll
                    for (int rho = 0; rho < 32; ++rho) v[rho] = s_ld_scratch(scr + P::p2_scratch(tid, s1, rho), pol_keep);
                }
                preloaded = false;
                P::template p2_math<true>(tid, tw, v);
                __syncthreads();             // the previous strip's X1 readers are done
                P::p2_store(tid, E, v);
                __syncthreads();
                P::p1_load(tid, E, v);
                dft<32, +1>(v);
                float2 *dst = A.c_out + fbase + (size_t)r_lo * M + s1 * WC + col_l;
                if (PIPE && s1 + CS >= C::NSTR && i + nclusters < A.K) {
                    const float2 *cin = A.c_in + (size_t)(i + nclusters) * M * M + (size_t)r_lo * M + crank * WC + col_l;
#pragma unroll
                    for (int k = 0; k < 32; ++k) {
                        st_stream(dst + (size_t)k * (NLO * M), v[k]);
                        v[k] = ld_stream(cin + (size_t)k * (NLO * M));
                    }
                    preloaded = true;
                } else if (PIPE && s1 + CS < C::NSTR) {
#pragma unroll
                    for (int k = 0; k < 32; ++k) {
                        st_stream(dst + (size_t)k * (NLO * M), v[k]);
                        v[k] = s_ld_scratch(scr + P::p2_scratch(tid, s1 + CS, k), pol_keep);
                    }
                    preloaded = true;
                } else {
#pragma unroll
                    for (int k = 0; k < 32; ++k) st_stream(dst + (size_t)k * (NLO * M), v[k]);
                }
            }
        }
    }

    if constexpr (MODE == FRAME_ERR) frame_err_reduce(s_a, s_q, s_d, smem_raw, C::NW, A.err_partials);
}

#endif  // __CUDACC__

}  // namespace sharp
