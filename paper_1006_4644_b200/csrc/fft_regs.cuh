// fft_regs.cuh -- in-register inverse DFTs and twiddle helpers for the sm_100a FFT passes.
//
// Everything here is the unnormalised INVERSE transform y_q = sum_r x_r e^{+2 pi i rq/R}
// (the e^{+2 pi i f t} of eq. 2.1).  The forward transform of load_segment is
// obtained from it by conjugation.  No code is shared with oracle/.
#pragma once
#include <cuda_runtime.h>

namespace cbmf {

__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 csqr(float2 a)
{
    return make_float2(fmaf(a.x, a.x, -a.y * a.y), 2.0f * a.x * a.y);
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }

// cos(2 pi a / 32), a = 0..8, correctly rounded to float.
__device__ __forceinline__ constexpr float cos32_table(int a)
{
    return a == 0 ? 1.0f
         : a == 1 ? 0.98078528040323044913f
         : a == 2 ? 0.92387953251128675613f
         : a == 3 ? 0.83146961230254523708f
         : a == 4 ? 0.70710678118654752440f
         : a == 5 ? 0.55557023301960222474f
         : a == 6 ? 0.38268343236508977173f
         : a == 7 ? 0.19509032201612826785f
         : 0.0f;
}

// x * e^{+2 pi i q / R}, 0 <= q < R/2, R a power of two <= 32; q and R are compile-time
// constants after unrolling, so the branches fold away.
template <int R>
__device__ __forceinline__ float2 twmul(float2 x, int q)
{
    const int a = q * (32 / R);                 // angle index, 0..15
    if (a == 0) return x;
    if (a == 8) return make_float2(-x.y, x.x);  // * i
    const float c = (a <= 8) ? cos32_table(a) : -cos32_table(16 - a);
    const float s = (a <= 8) ? cos32_table(8 - a) : cos32_table(a - 8);
    return make_float2(fmaf(x.x, c, -x.y * s), fmaf(x.x, s, x.y * c));
}

// Butterfly lo = e + o w, hi = e - o w with w = e^{+2 pi i q / R}, 0 <= q < R/2 (compile-time
// after unrolling).  Non-trivial twiddles are folded into FMAs: lo = e + o w costs four FFMA
// and hi = 2e - lo two more (6 instead of 8 instructions); w = (+-1 +- i)/sqrt 2 costs 2 FADD +
// 4 FFMA with no doubling.
template <int R>
__device__ __forceinline__ void bfly(const float2 e, const float2 o, const int q, float2& lo, float2& hi)
{
    const int a = q * (32 / R);                 // angle index, 0..15
    if (a == 0) {
        lo = cadd(e, o); hi = csub(e, o);
    } else if (a == 8) {                        // w = i
        lo = make_float2(e.x - o.y, e.y + o.x); hi = make_float2(e.x + o.y, e.y - o.x);
    } else if (a == 4) {                        // w = (1 + i) c
        const float c = cos32_table(4);
        const float dx = o.x - o.y, dy = o.x + o.y;
        lo = make_float2(fmaf(c, dx, e.x), fmaf(c, dy, e.y));
        hi = make_float2(fmaf(-c, dx, e.x), fmaf(-c, dy, e.y));
    } else if (a == 12) {                       // w = (-1 + i) c
        const float c = cos32_table(4);
        const float dx = o.x + o.y, dy = o.x - o.y;
        lo = make_float2(fmaf(-c, dx, e.x), fmaf(c, dy, e.y));
        hi = make_float2(fmaf(c, dx, e.x), fmaf(-c, dy, e.y));
    } else {
        const float c = (a <= 8) ? cos32_table(a) : -cos32_table(16 - a);
        const float s = (a <= 8) ? cos32_table(8 - a) : cos32_table(a - 8);
        lo = make_float2(fmaf(-o.y, s, fmaf(o.x, c, e.x)), fmaf(o.y, c, fmaf(o.x, s, e.y)));
        hi = make_float2(fmaf(2.0f, e.x, -lo.x), fmaf(2.0f, e.y, -lo.y));
    }
}

// Radix-R inverse DFT in registers, natural order in and out, decimation in time.
// NZ: only inputs v[0..NZ) are non-zero (the rest are never read), which prunes the leaves.
template <int R, int NZ>
struct DftP {
    static __device__ __forceinline__ void run(float2 (&v)[R])
    {
        if constexpr (NZ <= 1) {
#pragma unroll
            for (int q = 1; q < R; ++q) v[q] = v[0];
        } else {
            constexpr int H = R / 2;
            constexpr int NZE = ((NZ + 1) / 2 < H) ? (NZ + 1) / 2 : H;
            constexpr int NZO = (NZ / 2 < H) ? NZ / 2 : H;
            float2 e[H], o[H];
#pragma unroll
            for (int i = 0; i < H; ++i) { e[i] = v[2 * i]; o[i] = v[2 * i + 1]; }
            DftP<H, NZE>::run(e);
            DftP<H, NZO>::run(o);
#pragma unroll
            for (int q = 0; q < H; ++q) bfly<R>(e[q], o[q], q, v[q], v[q + H]);
        }
    }
};
template <int NZ>
struct DftP<1, NZ> {
    static __device__ __forceinline__ void run(float2 (&)[1]) {}
};

template <int R>
__device__ __forceinline__ void dft(float2 (&v)[R]) { DftP<R, R>::run(v); }

// e^{+2 pi i num/den} with den a power of two <= 2^24 and 0 <= num < den: the argument of
// sincospif is formed exactly (integers below 2^24 and a power-of-two scale).
__device__ __forceinline__ float2 expi_frac(int num, float two_over_den)
{
    float s, c;
    sincospif((float)num * two_over_den, &s, &c);
    return make_float2(c, s);
}

// x[r] *= base * g^r for r = 0..R-1 (r = 0 multiplies by base only when HAS_BASE).
// Powers are built as g^(8 hi) * (base g^lo): every factor is at most 6 roundings deep.
template <int R, bool HAS_BASE>
__device__ __forceinline__ void mul_powers(float2 (&x)[R], float2 g, float2 base)
{
    constexpr int LO = (R < 8) ? R : 8;
    float2 pl[LO];
    const float2 g2 = csqr(g);
    if constexpr (HAS_BASE) {
        pl[0] = base;
        pl[1] = cmul(base, g);
    } else {
        pl[0] = make_float2(1.0f, 0.0f);
        pl[1] = g;
    }
    if constexpr (LO > 2) {
        const float2 g4 = csqr(g2);
        pl[2] = HAS_BASE ? cmul(pl[0], g2) : g2;
        pl[3] = cmul(pl[1], g2);
        if constexpr (LO > 4) {
            pl[4] = HAS_BASE ? cmul(pl[0], g4) : g4;
            pl[5] = cmul(pl[1], g4);
            pl[6] = cmul(pl[2], g4);
            pl[7] = cmul(pl[3], g4);
        }
        if constexpr (R > 8) {
            const float2 g8 = csqr(g4);
            float2 ph = g8;
#pragma unroll
            for (int hi = 1; hi < R / 8; ++hi) {
#pragma unroll
                for (int lo = 0; lo < 8; ++lo) x[8 * hi + lo] = cmul(x[8 * hi + lo], cmul(pl[lo], ph));
                if (hi + 1 < R / 8) ph = (hi == 1) ? csqr(g8) : cmul(ph, g8);
            }
        }
    }
#pragma unroll
    for (int lo = (HAS_BASE ? 0 : 1); lo < LO; ++lo) x[lo] = cmul(x[lo], pl[lo]);
}

}  // namespace cbmf
