// frame_common.cuh -- what every variant of the fused per-frame kernel shares: the modes, the argument block and
// the global-memory access helpers.
#pragma once
#include "fft_regs.cuh"

namespace sharp {

enum FrameMode : int {
    FRAME_ITER = 0,  // c_out = beta z + (1-2 beta) P_a z
    FRAME_FFT = 1,   // c_out = F z  in natural (u,v) order, unitary (test hook)
    FRAME_ERR = 2    // no output; accumulates ||P_a z - z||^2, ||P_Q z - z||^2, ||z - z_prev||^2
};

struct DevScalars {
    double A2;       // ||a||^2 = sum I          (reading G12)
    float thr2;      // (m * thr)^2, thr = 1e-4 a_rms: threshold on |Z^|^2 (reading G4)
    float pad;
};

struct FrameArgs {
    const float2 *c_in;      // K m m   frame-local state (or the operand of the op_* hooks)
    float2 *c_out;           // K m m
    const float *a_int;      // K m m   amplitudes / m in position space
    const float2 *psi_v;     // object; may be NULL (z = c_in)
    const float2 *w_form;    // m m
    const int *pos;          // K x 2
    float2 *scratch;         // gridDim.x * m * m
    int *sched, *sched_next; // frame counters of the dynamic schedule: this launch's (zero on entry), and the one it zeroes for the next launch
    const DevScalars *sc;
    int K, nr, nc;           // frames, object rows / columns (nr: only the periodic wrap and FRAME_ERR need it)
    float bm;                // beta / m^2
    float om;                // 1 - 2 beta
    int conj_io;             // FRAME_FFT: conjugate input and output (gives F*)
    // FRAME_ERR only
    const float2 *c_prev, *psi_v_prev, *w_form_prev;   // previous iterate in factored form (c_prev NULL: z_prev = 0)
    const float2 *psi_z, *w_cur;                        // P_Q z = w_cur . T psi_z
    double *err_partials;                               // gridDim.x * 3
};

#if defined(__CUDACC__)
__device__ __forceinline__ float2 ld_stream(const float2 *p) { return __ldcs(p); }
__device__ __forceinline__ void st_stream(float2 *p, float2 v) { __stcs(p, v); }
__device__ __forceinline__ float2 ld_l2(const float2 *p) { return __ldcg(p); }
__device__ __forceinline__ void st_l2(float2 *p, float2 v) { __stcg(p, v); }

__device__ __forceinline__ void prefetch_l2_bulk(const void *p, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// Tensor memory (TMEM, 256 KB per SM, otherwise idle here) as a per-thread store for the probe values a thread needs
// for every frame: written once per launch with tcgen05.st into the thread's own TMEM lane, read back with tcgen05.ld.
__device__ __forceinline__ unsigned r_smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void r_tmem_alloc(unsigned *smem_slot, int ncols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(r_smem_u32(smem_slot)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void r_tmem_dealloc(unsigned taddr, int ncols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void r_tmem_st16(unsigned taddr, const float2 *x)   // 8 complex -> 16 columns
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
                 ::"r"(taddr), "f"(x[0].x), "f"(x[0].y), "f"(x[1].x), "f"(x[1].y), "f"(x[2].x), "f"(x[2].y), "f"(x[3].x),
                 "f"(x[3].y), "f"(x[4].x), "f"(x[4].y), "f"(x[5].x), "f"(x[5].y), "f"(x[6].x), "f"(x[6].y), "f"(x[7].x), "f"(x[7].y)
                 : "memory");
}
__device__ __forceinline__ void r_tmem_ld16(unsigned taddr, float2 *x)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=f"(x[0].x), "=f"(x[0].y), "=f"(x[1].x), "=f"(x[1].y), "=f"(x[2].x), "=f"(x[2].y), "=f"(x[3].x), "=f"(x[3].y),
                   "=f"(x[4].x), "=f"(x[4].y), "=f"(x[5].x), "=f"(x[5].y), "=f"(x[6].x), "=f"(x[6].y), "=f"(x[7].x), "=f"(x[7].y)
                 : "r"(taddr)
                 : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Cluster helpers: the CS CTAs of a thread-block cluster share one frame (and one L2 scratch slot); strips are
// dealt round-robin by cluster rank and the three stage changes are cluster barriers (release/acquire, so the
// L2-resident scratch written with st.cg by one CTA is visible to the ld.cg of the others).
__device__ __forceinline__ unsigned cluster_rank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_barrier()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// ---- arithmetic both frame kernels share (written once) --------------------------------------------------------------
// Magnitude projection fused with the frame half of RAAR, on 8 Fourier coefficients x[] (un-normalised transform) with
// their amplitudes av[] = a/m:  C^ = Z^ (beta/m^2 + (1 - 2 beta)(a/m)/|Z^|);  |Z^|^2 <= thr2 takes the phase as 1 (reading G4).
__device__ __forceinline__ void frame_project8(float2 *x, const float *av, float thr2, float bm, float om)
{
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const float mag2 = x[k].x * x[k].x + x[k].y * x[k].y;
        const float oa = om * av[k];
        if (mag2 > thr2) {
            const float sc = fmaf(oa, rsqrtf(mag2), bm);
            x[k].x *= sc;
            x[k].y *= sc;
        } else {
            x[k].x = fmaf(bm, x[k].x, oa);
            x[k].y = bm * x[k].y;
        }
    }
}

// sum over a thread's 32 coefficients of |a - |F z||^2 (= |P_a z - z|^2 by Parseval; G4 branch: |a - F z|^2); ap points at
// the thread's first amplitude, consecutive registers are 32 floats apart
template <int M>
__device__ __forceinline__ float frame_err_a32(const float2 *v, const float *ap, float thr2)
{
    const float fm = (float)M, inv_m = 1.0f / (float)M;
    float sa = 0.f;
#pragma unroll
    for (int q = 0; q < 32; ++q) {
        const float a = __ldcs(ap + q * 32) * fm;
        const float mag2 = v[q].x * v[q].x + v[q].y * v[q].y;
        if (mag2 > thr2) {
            const float d = a - sqrtf(mag2) * inv_m;
            sa += d * d;
        } else {
            const float dx = a - v[q].x * inv_m, dy = v[q].y * inv_m;
            sa += dx * dx + dy * dy;
        }
    }
    return sa;
}

// |P_Q z - z|^2 and |z - z_prev|^2 over a thread's 32 frame pixels (rows r_lo + NLO k of column col); v[] holds z.
// Four pixels at a time: all loads of a batch are issued before its arithmetic (up to 20 per batch; eight spill), and the cases
// (no previous iterate / previous iterate without an object part) are decided outside the loops.
template <int M, int NLO>
__device__ __forceinline__ void frame_err_qd32(const FrameArgs &A, const float2 *v, size_t fbase, int xr, int xc, int r_lo, int col,
                                                float &sq, float &sd)
{
    sq = 0.f;
    sd = 0.f;
    int pcw = xc + col;                        // modulo the image size (identity without the periodic boundary)
    if (pcw >= A.nc) pcw -= A.nc;
    const bool have_prev = A.c_prev != nullptr, have_pv = have_prev && A.psi_v_prev != nullptr;
#pragma unroll
    for (int k0 = 0; k0 < 32; k0 += 4) {
        float2 wc[4], pz[4], cp[4], wp[4], pp[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int r = r_lo + NLO * (k0 + j);
            int prw = xr + r;
            if (prw >= A.nr) prw -= A.nr;
            const size_t op = (size_t)prw * A.nc + pcw;
            wc[j] = __ldg(A.w_cur + r * M + col);
            pz[j] = __ldg(A.psi_z + op);
            cp[j] = have_prev ? ld_stream(A.c_prev + fbase + (size_t)r * M + col) : make_float2(0.f, 0.f);
            wp[j] = have_pv ? __ldg(A.w_form_prev + r * M + col) : make_float2(0.f, 0.f);
            pp[j] = have_pv ? __ldg(A.psi_v_prev + op) : make_float2(0.f, 0.f);
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float2 d = csub(cmul(wc[j], pz[j]), v[k0 + j]);
            sq += d.x * d.x + d.y * d.y;
            const float2 zp = cadd(cp[j], cmul(wp[j], pp[j]));      // z_prev = c_prev + w_form_prev . T psi_v_prev (0 if absent)
            const float2 dd = csub(v[k0 + j], zp);
            sd += dd.x * dd.x + dd.y * dd.y;
        }
    }
}

// deterministic reduction of the three residual sums of a CTA: fixed xor-tree inside each warp (shuffles), then the
// warp sums in warp order by thread 0; one triple per CTA
__device__ __forceinline__ void frame_err_reduce(double s_a, double s_q, double s_d, unsigned char *smem_raw, int nwarps,
                                                  double *err_partials)
{
    const int tid = threadIdx.x, wq = tid >> 5, lane = tid & 31;
    __syncthreads();
    double *red = reinterpret_cast<double *>(smem_raw);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        s_a += __shfl_xor_sync(0xffffffffu, s_a, off);
        s_q += __shfl_xor_sync(0xffffffffu, s_q, off);
        s_d += __shfl_xor_sync(0xffffffffu, s_d, off);
    }
    if (lane == 0) {
        red[3 * wq + 0] = s_a;
        red[3 * wq + 1] = s_q;
        red[3 * wq + 2] = s_d;
    }
    __syncthreads();
    if (tid == 0) {
        double a = 0.0, q = 0.0, d = 0.0;
        for (int w = 0; w < nwarps; ++w) {
            a += red[3 * w + 0];
            q += red[3 * w + 1];
            d += red[3 * w + 2];
        }
        err_partials[3 * blockIdx.x + 0] = a;
        err_partials[3 * blockIdx.x + 1] = q;
        err_partials[3 * blockIdx.x + 2] = d;
    }
}

#endif  // __CUDACC__


}  // namespace sharp
