// overlap_tma.cuh -- a5 overlap (Eq. 8-9) in gather form with the tile/frame intersections
// fetched by the TMA unit (cp.async.bulk.tensor), for the two modes on the iteration path (OV_ITER, OV_L).
//
// Same sum, same order and same epilogue as k_overlap (object_kernels.cuh): one CTA per 32 x 32 object tile, the
// tile's CSR list of covering frames in ascending index, num(p) = sum_i conj(w(p - x_i)) f_i(p - x_i).  What
// differs is the data path: for frame i the 32 x 32 box of f_i at frame coordinates (tile origin - x_i) is one
// 3-D tensor copy (x, y, frame) and the matching box of w one 2-D copy; coordinates outside the frame are
// zero-filled by the hardware, so no thread is predicated off and the partial intersections cost no branches.
// STAGES boxes are in flight per CTA (mbarrier per stage); the loads never occupy registers or the L1 miss path,
// which is what limited the register-gather version (profiles/r01_summary.md).
#pragma once
#include <cuda.h>
#include <cstdio>

#include "object_kernels.cuh"
#include "frame_ws.cuh"   // mbarrier helpers

namespace sharp {

constexpr int OVT_STAGES = 6;
// The box is 34 pixels wide and starts at an even frame column: the TMA unit faults on box origins whose byte
// address is not a multiple of 16 (observed on sm_100a: odd x with 8-byte elements), so the odd case reads one
// column to the left and the threads index with the parity offset.
constexpr int OVT_BOXW = TILE + 2;
constexpr int OVT_BOX_BYTES = OVT_BOXW * TILE * 8;                   // 8.5 KB per box
constexpr int OVT_SMEM_BYTES = OVT_STAGES * 2 * OVT_BOX_BYTES + 128;
static_assert(OVT_BOX_BYTES % 128 == 0, "boxes must stay 128-byte aligned");   // f and w boxes + barriers

__device__ __forceinline__ void mbar_expect_tx(void *bar, unsigned bytes)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int x, int y, int z, void *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
            smem_u32(dst)),
        "l"(reinterpret_cast<unsigned long long>(map)), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void tma_load_2d(void *dst, const CUtensorMap *map, int x, int y, void *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
            smem_u32(dst)),
        "l"(reinterpret_cast<unsigned long long>(map)), "r"(x), "r"(y), "r"(smem_u32(bar))
        : "memory");
}

template <int MODE>
__global__ void __launch_bounds__(256) k_overlap_tma(OverlapArgs A, const __grid_constant__ CUtensorMap mapF,
                                                      const __grid_constant__ CUtensorMap mapW)
{
    static_assert(MODE == OV_ITER || MODE == OV_L, "TMA overlap serves the iteration-path modes");
    extern __shared__ __align__(128) unsigned char ov_smem[];
    float2 *boxF = reinterpret_cast<float2 *>(ov_smem);
    float2 *boxW = reinterpret_cast<float2 *>(ov_smem + OVT_STAGES * OVT_BOX_BYTES);
    unsigned long long *full = reinterpret_cast<unsigned long long *>(ov_smem + 2 * OVT_STAGES * OVT_BOX_BYTES);
    int *s_odd = reinterpret_cast<int *>(full + OVT_STAGES);   // parity of the box origin, per stage

    const int tile = blockIdx.x;
    const int tr = tile / A.tiles_c, tc = tile % A.tiles_c;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int pc = tc * TILE + tx;
    const int pr0 = tr * TILE + ty;
    const int beg = A.tile_ptr[tile], end = A.tile_ptr[tile + 1];
    const int n = end - beg;

    if (threadIdx.x == 0) {
        for (int s = 0; s < OVT_STAGES; ++s) mbar_init(full + s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    auto issue = [&](int e) {   // thread 0 only: boxes of list entry e into stage e % STAGES
        const int s = e % OVT_STAGES;
        const int fi = __ldg(A.tile_frames + beg + e);
        const int x = tc * TILE - __ldg(A.pos + 2 * fi + 1), y = tr * TILE - __ldg(A.pos + 2 * fi);
        s_odd[s] = x & 1;                              // published by the release of the arrive below
        mbar_expect_tx(full + s, 2 * OVT_BOX_BYTES);
        tma_load_3d(boxF + s * (OVT_BOXW * TILE), &mapF, x & ~1, y, fi, full + s);
        tma_load_2d(boxW + s * (OVT_BOXW * TILE), &mapW, x & ~1, y, full + s);
    };
    if (threadIdx.x == 0)
        for (int e = 0; e < min(n, OVT_STAGES); ++e) issue(e);

    float2 num[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) num[k] = make_float2(0.f, 0.f);

    for (int e = 0; e < n; ++e) {
        const int s = e % OVT_STAGES;
        {
            unsigned spins = 0;
            while (!mbar_try_wait(full + s, (unsigned)((e / OVT_STAGES) & 1))) {
                if (++spins > (1u << 22)) {
                    __trap();   // protocol error: surface as a launch failure, never hang
                }
            }
        }
        const int odd = s_odd[s];
        const float2 *bf = boxF + s * (OVT_BOXW * TILE) + odd, *bw = boxW + s * (OVT_BOXW * TILE) + odd;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float2 w_ = bw[(ty + 8 * k) * OVT_BOXW + tx], f_ = bf[(ty + 8 * k) * OVT_BOXW + tx];
            num[k].x += w_.x * f_.x + w_.y * f_.y;   // conj(w) f; zero outside the frame
            num[k].y += w_.x * f_.y - w_.y * f_.x;
        }
        __syncthreads();                             // every thread is done with stage s
        if (threadIdx.x == 0 && e + OVT_STAGES < n) issue(e + OVT_STAGES);
    }

    if (pc >= A.nc) return;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int pr = pr0 + 8 * k;
        if (pr >= A.nr) continue;
        const size_t p = (size_t)pr * A.nc + pc;
        const float d = A.den[p];
        const bool lit = d > 0.f;
        if constexpr (MODE == OV_L) {
            A.out[p] = lit ? make_float2(num[k].x / d, num[k].y / d) : make_float2(0.f, 0.f);
        } else {
            float2 py = make_float2(0.f, 0.f), pv = py;
            if (lit) {
                const float2 pz = A.psi_z[p];
                const float inv = 1.0f / (1.0f - 2.0f * A.beta);
                py.x = (num[k].x / d - A.beta * pz.x) * inv;
                py.y = (num[k].y / d - A.beta * pz.y) * inv;
                pv.x = A.beta * (2.0f * py.x - pz.x);
                pv.y = A.beta * (2.0f * py.y - pz.y);
            }
            A.psi_z[p] = py;
            A.psi_v_out[p] = pv;
        }
    }
}

}  // namespace sharp
