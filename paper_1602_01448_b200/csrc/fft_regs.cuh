// fft_regs.cuh -- in-register radix-R DFT butterflies (R = 2, 4, 8, 16, 32) for the fused frame kernel.
//
// dft<R, SGN>(x): x[k] <- sum_n x[n] exp(SGN * 2 pi i n k / R), natural order in and out, un-normalised.
// SGN = -1 is the forward kernel of Eq. (2) under reading G2, SGN = +1 its adjoint.
// Everything is compile-time indexed so that x[] lives in registers; composite sizes use the Cooley-Tukey
// split R = R1 * R2 (n = R2 n1 + n2, k = k1 + R1 k2) with constant twiddles from a 32-point table.
#pragma once
#include <cuda_runtime.h>
#include <utility>

#define SHARP_HD __host__ __device__ __forceinline__

namespace sharp {

// cos / sin of 2 pi e / 32, e in [0, 32), from the first-octant values (correctly rounded literals).
SHARP_HD constexpr float w32_cos_oct(int e)  // e in [0, 8]
{
    return e == 0 ? 1.0f : e == 1 ? 0.98078528040323044913f : e == 2 ? 0.92387953251128675613f
         : e == 3 ? 0.83146961230254523708f : e == 4 ? 0.70710678118654752440f : e == 5 ? 0.55557023301960222474f
         : e == 6 ? 0.38268343236508977173f : e == 7 ? 0.19509032201612826785f : 0.0f;
}
SHARP_HD constexpr float w32_cos(int e)
{
    e &= 31;
    return e <= 8 ? w32_cos_oct(e) : e <= 16 ? -w32_cos_oct(16 - e) : e <= 24 ? -w32_cos_oct(e - 16) : w32_cos_oct(32 - e);
}
SHARP_HD constexpr float w32_sin(int e) { return w32_cos(e - 8); }

// Complex add / subtract as ONE packed instruction on sm_100a (add.f32x2 / sub.f32x2 -> FADD2): the butterflies are
// mostly these, and the passes are issue-slot bound, so halving their instruction count matters; each component is
// still one IEEE round-to-nearest add (the only numerical difference to the scalar form is that the compiler can no
// longer contract such an add with a neighbouring multiply into an FMA).
SHARP_HD float2 cadd(float2 a, float2 b)
{
#if defined(__CUDA_ARCH__) && __CUDA_ARCH__ >= 1000 && !defined(SHARP_NO_PACKED_F32)
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(*reinterpret_cast<unsigned long long *>(&a)), "l"(*reinterpret_cast<unsigned long long *>(&b)));
    return *reinterpret_cast<float2 *>(&d);
#else
    return make_float2(a.x + b.x, a.y + b.y);
#endif
}
SHARP_HD float2 csub(float2 a, float2 b)
{
#if defined(__CUDA_ARCH__) && __CUDA_ARCH__ >= 1000 && !defined(SHARP_NO_PACKED_F32)
    unsigned long long d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(*reinterpret_cast<unsigned long long *>(&a)), "l"(*reinterpret_cast<unsigned long long *>(&b)));
    return *reinterpret_cast<float2 *>(&d);
#else
    return make_float2(a.x - b.x, a.y - b.y);
#endif
}
SHARP_HD float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// a * conj(b)
SHARP_HD float2 cmulc(float2 a, float2 b) { return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }

// a * exp(SGN * 2 pi i * E / 32)
template <int E, int SGN>
SHARP_HD float2 cmul_w32(float2 a)
{
    constexpr int e = ((E % 32) + 32) % 32;
    if constexpr (e == 0) return a;
    else if constexpr (e == 16) return make_float2(-a.x, -a.y);
    else if constexpr (e == 8) return SGN > 0 ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
    else if constexpr (e == 24) return SGN > 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
    else {
        constexpr float c = w32_cos(e);
        constexpr float s = (SGN > 0 ? 1.0f : -1.0f) * w32_sin(e);
        return make_float2(a.x * c - a.y * s, a.x * s + a.y * c);
    }
}

template <int R, int SGN, int STRIDE>
struct Dft;

template <int SGN, int STRIDE>
struct Dft<2, SGN, STRIDE> {
    static SHARP_HD void run(float2 *x)
    {
        float2 a = x[0], b = x[STRIDE];
        x[0] = cadd(a, b);
        x[STRIDE] = csub(a, b);
    }
};

template <int SGN, int STRIDE>
struct Dft<4, SGN, STRIDE> {
    static SHARP_HD void run(float2 *x)
    {
        float2 a0 = x[0], a1 = x[STRIDE], a2 = x[2 * STRIDE], a3 = x[3 * STRIDE];
        float2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3);
        float2 t3 = cmul_w32<8, SGN>(csub(a1, a3));  // (a1 - a3) * (SGN i)
        x[0] = cadd(t0, t2);
        x[STRIDE] = cadd(t1, t3);
        x[2 * STRIDE] = csub(t0, t2);
        x[3 * STRIDE] = csub(t1, t3);
    }
};

// Composite R = R1 * R2.
template <int R, int R1, int R2, int SGN, int STRIDE>
struct DftSplit {
    template <int N2, int K1>
    static SHARP_HD void twiddle_one(float2 *x)
    {
        x[(R2 * K1 + N2) * STRIDE] = cmul_w32<(N2 * K1) * (32 / R), SGN>(x[(R2 * K1 + N2) * STRIDE]);
    }
    template <int N2, int... K1s>
    static SHARP_HD void twiddle_row(float2 *x, std::integer_sequence<int, K1s...>)
    {
        (twiddle_one<N2, K1s>(x), ...);
    }
    template <int... N2s>
    static SHARP_HD void twiddle_all(float2 *x, std::integer_sequence<int, N2s...>)
    {
        (twiddle_row<N2s>(x, std::make_integer_sequence<int, R1>{}), ...);
    }
    static SHARP_HD void run(float2 *x)
    {
        // R1-point DFTs over n1 (elements R2 n1 + n2), in place: A[k1][n2] at R2 k1 + n2
#pragma unroll
        for (int n2 = 0; n2 < R2; ++n2) Dft<R1, SGN, R2 * STRIDE>::run(x + n2 * STRIDE);
        twiddle_all(x, std::make_integer_sequence<int, R2>{});
        // R2-point DFTs over n2 for each k1: X[k1 + R1 k2] at R2 k1 + k2
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) Dft<R2, SGN, STRIDE>::run(x + R2 * k1 * STRIDE);
        // back to natural order: out[k1 + R1 k2] = x[R2 k1 + k2]
        float2 t[R];
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1)
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) t[k1 + R1 * k2] = x[(R2 * k1 + k2) * STRIDE];
#pragma unroll
        for (int k = 0; k < R; ++k) x[k * STRIDE] = t[k];
    }
};

template <int SGN, int STRIDE>
struct Dft<8, SGN, STRIDE> : DftSplit<8, 4, 2, SGN, STRIDE> {};
template <int SGN, int STRIDE>
struct Dft<16, SGN, STRIDE> : DftSplit<16, 4, 4, SGN, STRIDE> {};
template <int SGN, int STRIDE>
struct Dft<32, SGN, STRIDE> : DftSplit<32, 8, 4, SGN, STRIDE> {};

template <int R, int SGN>
SHARP_HD void dft(float2 *x)
{
    Dft<R, SGN, 1>::run(x);
}

}  // namespace sharp
