// probe_kernels.cuh -- the small kernels of SURVEY.md section 8(f) rows 1 and 3: the error against a known solution
// (Eq. 14), the default initialisations (steps 2-3 of the reconstruction sequence), the illumination Fourier
// constraints and the centre-of-mass re-centring (step 7).  All of them work on one m x m probe or on object-sized
// arrays; the two m x m Fourier transforms they need are launches of the fused frame kernel in FRAME_FFT mode with
// K = 1 (sharp_b200.cu), so there is one FFT implementation in the library.
#pragma once
#include "frame_common.cuh"
#include "object_kernels.cuh"

namespace sharp {

// fixed-tree block reduction of NV doubles per thread (256 threads); result valid in thread 0
template <int NV>
__device__ __forceinline__ void block_reduce_256(double (&v)[NV], double *red /* 8 * NV doubles of shared memory */)
{
    const int lane = threadIdx.x & 31, wq = threadIdx.x >> 5;
#pragma unroll
    for (int j = 0; j < NV; ++j)
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v[j] += __shfl_xor_sync(0xffffffffu, v[j], off);
    if (lane == 0)
#pragma unroll
        for (int j = 0; j < NV; ++j) red[wq * NV + j] = v[j];
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            double s = 0.0;
            for (int w = 0; w < 8; ++w) s += red[w * NV + j];
            v[j] = s;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// Eq. (14):  eps_0 = min_phi || Q*(e^{i phi} z - z_0) || / || Q* z_0 ||,  z_0 = Q_{w0} psi_0.
// With A = Q* z and B = Q* z_0 the minimum over the global phase is ||A||^2 + ||B||^2 - 2 |<B, A>|.
//   A(p) = psi_z(p) den(p)                          (psi_z = Q*z / Q*Q is the maintained object estimate, den = Q*Q)
//   B(p) = psi_0(p) sum_i conj(w(p-x_i)) w0(p-x_i)  (= psi_0 den when w0 is the current illumination; `cross` otherwise)
// Per-block partial sums (||A||^2, ||B||^2, Re<B,A>, Im<B,A>) in double, fixed order; k_sum_quads finishes them.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_eps0_partial(size_t n, const float2 *psi_z, const float *den, const float2 *psi0,
                                                       const float2 *cross, double *partials)
{
    double v[4] = {0.0, 0.0, 0.0, 0.0};
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < n; g += (size_t)gridDim.x * blockDim.x) {
        const float d = den[g];
        const float2 pz = psi_z[g], p0 = psi0[g];
        const float2 a = make_float2(pz.x * d, pz.y * d);
        const float2 b = cross != nullptr ? cmul(p0, cross[g]) : make_float2(p0.x * d, p0.y * d);
        v[0] += (double)a.x * a.x + (double)a.y * a.y;
        v[1] += (double)b.x * b.x + (double)b.y * b.y;
        v[2] += (double)b.x * a.x + (double)b.y * a.y;      // conj(b) a
        v[3] += (double)b.x * a.y - (double)b.y * a.x;
    }
    __shared__ double red[32];
    block_reduce_256<4>(v, red);
    if (threadIdx.x == 0)
        for (int j = 0; j < 4; ++j) partials[4 * blockIdx.x + j] = v[j];
}

__global__ void k_sum_quads(int n, const double *partials, double *out)
{
    if (threadIdx.x < 4 && blockIdx.x == 0) {
        double s = 0.0;
        for (int j = 0; j < n; ++j) s += partials[4 * j + threadIdx.x];
        out[threadIdx.x] = s;
    }
}

// ---------------------------------------------------------------------------------------------------------
// Step 2: w0 = F*( sqrt(average frame) ).  The average runs over the stored amplitudes (a/m in slot
// order, see k_amplitudes): mean_i I_i = (m^2/K) sum_i a_int^2.  Two stages in double, fixed order (chunks of
// consecutive frames, then the chunks in ascending order); the result is written in natural (u,v) order as a complex
// array for the inverse transform.  k_cyclic_shift then moves the result to the frame centre (reading G21).
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_mean_frame_partial(int m, int K, int chunk, const float *a_int, double *part)
{
    const int slot = blockIdx.x * blockDim.x + threadIdx.x;
    const size_t mm = (size_t)m * m;
    const int i0 = blockIdx.y * chunk, i1 = min(K, i0 + chunk);
    double s = 0.0;
    for (int i = i0; i < i1; ++i) {
        const float a = __ldcs(a_int + (size_t)i * mm + slot);
        s += (double)a * (double)a;
    }
    part[(size_t)blockIdx.y * mm + slot] = s;
}

// chunks -> part[0 .. m*m) in ascending chunk order (each thread reads and then writes only its own slot)
__global__ void __launch_bounds__(256) k_mean_frame_sum(int m, int nchunks, double *part)
{
    const int slot = blockIdx.x * blockDim.x + threadIdx.x;
    const size_t mm = (size_t)m * m;
    double s = 0.0;
    for (int j = 0; j < nchunks; ++j) s += part[(size_t)j * mm + slot];
    part[slot] = s;
}

// K = the frames of the WHOLE scan (a sharded plan sums part[] over its ranks first)
__global__ void __launch_bounds__(256) k_mean_frame_sqrt(int m, long long K, const double *part, float2 *abar)
{
    const int slot = blockIdx.x * blockDim.x + threadIdx.x;
    const size_t mm = (size_t)m * m;
    int u, v;
    amp_slot_freq(m, slot, u, v);
    abar[(size_t)u * m + v] = make_float2((float)sqrt(part[slot] * (double)mm / (double)K), 0.f);
}

// out[(r + d_r) mod m][(c + d_c) mod m] = in[r][c];  the shift is read from device memory (written by k_probe_moments)
// or, when `shift` is NULL, is (m/2, m/2)
__global__ void __launch_bounds__(256) k_cyclic_shift(int m, const float2 *in, const int *shift, float2 *out)
{
    const int pix = blockIdx.x * blockDim.x + threadIdx.x;
    const int r = pix / m, c = pix % m;
    const int dr = shift ? shift[0] : m / 2, dc = shift ? shift[1] : m / 2;
    const int rr = ((r + dr) % m + m) % m, cc = ((c + dc) % m + m) % m;
    out[(size_t)rr * m + cc] = in[pix];
}

// ---------------------------------------------------------------------------------------------------------
// Step 3: psi0 ~ U[0,1).  Counter-based: splitmix64 of (splitmix64(seed) + pixel index), top 24 bits
// -> float in [0,1); imaginary part 0.  The oracle implements the same generator; the values are compared bit-exactly.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long splitmix64(unsigned long long x)
{
    x += 0x9E3779B97F4A7C15ULL;
    unsigned long long z = x;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

__global__ void __launch_bounds__(256) k_random_object(size_t n, unsigned long long seed, float2 *out)
{
    const unsigned long long k = splitmix64(seed);
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < n; g += (size_t)gridDim.x * blockDim.x)
        out[g] = make_float2((float)(splitmix64(k + g) >> 40) * (1.0f / 16777216.0f), 0.f);
}

// ---------------------------------------------------------------------------------------------------------
// Step 7 constraints, applied to W = F w in natural order (unitary):
//   kind 1  W <- W m_w                       (Fourier mask)
//   kind 2  W <- (W / |W|) a_w               (Fourier amplitude; |W| <= thr_w: W <- a_w, reading G24)
// k_constraint_scalars: thr_w^2 = (1e-4)^2 mean(a_w^2), one block, fixed order.
// ---------------------------------------------------------------------------------------------------------
struct ProbeScalars {
    float thr2;       // thr_w^2 for the amplitude constraint
    int shift[2];     // last re-centring shift (d_r, d_c)
    int total[2];     // sum of all shifts since the constraint / recentring was configured
};

__global__ void __launch_bounds__(256) k_constraint_scalars(int mm, const float *con, double tau, ProbeScalars *ps)
{
    double v[1] = {0.0};
    for (int g = threadIdx.x; g < mm; g += blockDim.x) v[0] += (double)con[g] * (double)con[g];
    __shared__ double red[8];
    block_reduce_256<1>(v, red);
    if (threadIdx.x == 0) ps->thr2 = (float)(tau * tau * v[0] / (double)mm);
}

__global__ void __launch_bounds__(256) k_probe_fourier(int mm, int kind, const float *con, const ProbeScalars *ps, float2 *W)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= mm) return;
    float2 x = W[q];
    const float cv = con[q];
    if (kind == 1) {
        x.x *= cv;
        x.y *= cv;
    } else {
        const float mag2 = x.x * x.x + x.y * x.y;
        if (mag2 > ps->thr2) {
            const float sc = cv * rsqrtf(mag2);
            x.x *= sc;
            x.y *= sc;
        } else {
            x = make_float2(cv, 0.f);
        }
    }
    W[q] = x;
}

// ---------------------------------------------------------------------------------------------------------
// Re-centring (readings G22, G23): centre of mass of |w|^2 over the frame indices, integer shift
// d = floor(m/2 - cm + 1/2) per axis.  One block of 256 threads, double accumulation, fixed order.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_probe_moments(int m, const float2 *w, ProbeScalars *ps)
{
    double v[3] = {0.0, 0.0, 0.0};
    for (int g = threadIdx.x; g < m * m; g += blockDim.x) {
        const float2 x = w[g];
        const double p = (double)x.x * x.x + (double)x.y * x.y;
        v[0] += p;
        v[1] += p * (double)(g / m);
        v[2] += p * (double)(g % m);
    }
    __shared__ double red[24];
    block_reduce_256<3>(v, red);
    if (threadIdx.x == 0) {
        int dr = 0, dc = 0;
        if (v[0] > 0.0) {
            dr = (int)floor((double)(m / 2) - v[1] / v[0] + 0.5);
            dc = (int)floor((double)(m / 2) - v[2] / v[0] + 0.5);
        }
        ps->shift[0] = dr;
        ps->shift[1] = dc;
        ps->total[0] += dr;
        ps->total[1] += dc;
    }
}

}  // namespace sharp
