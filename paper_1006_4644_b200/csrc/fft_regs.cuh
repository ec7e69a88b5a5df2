// fft_regs.cuh -- in-register inverse DFTs and twiddle helpers for the sm_100a FFT passes.
//
// Everything here is the unnormalised INVERSE transform y_q = sum_r x_r e^{+2 pi i rq/R}
// (the e^{+2 pi i f t} of eq. 2.1).  The forward transform of load_segment is
// obtained from it by conjugation.  No code is shared with oracle/.
//
// Complex numbers are PACKED: one 64-bit register pair (re in the low word, im in the high
// word), and the arithmetic is the sm_100 two-wide FP32 instructions (PTX add/mul/fma.f32x2,
// SASS FADD2 / FMUL2 / FFMA2).  A complex add is one instruction, a complex multiply two, a
// radix-2 butterfly with a general twiddle three; the swaps, broadcasts and per-half sign
// flips written below as pk(...) are operand modifiers of those instructions (.LO_HI, .F32,
// .NP), not extra moves.  The FP32 pipe time is that of the scalar code, the number of issue
// slots is half.
#pragma once
#include <cuda_runtime.h>

namespace cbmf {

typedef unsigned long long c2;            // packed complex float: (re, im)

__device__ __forceinline__ c2 pk(float x, float y)
{
    c2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y));
    return r;
}
__device__ __forceinline__ void unpk(c2 v, float& x, float& y)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(v));
}
__device__ __forceinline__ float re(c2 v) { float x, y; unpk(v, x, y); return x; }
__device__ __forceinline__ float im(c2 v) { float x, y; unpk(v, x, y); return y; }
__device__ __forceinline__ c2 bc(float s) { return pk(s, s); }
__device__ __forceinline__ c2 czero() { return 0ULL; }

__device__ __forceinline__ c2 add2(c2 a, c2 b)
{
    c2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ c2 sub2(c2 a, c2 b)
{
    c2 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ c2 mul2(c2 a, c2 b)
{
    c2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ c2 fma2(c2 a, c2 b, c2 c)
{
    c2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}

// a * w = a.x (w.x, w.y) + a.y (-w.y, w.x): FMUL2 + FFMA2 (the (-w.y, w.x) operand is the
// .LO_HI.NP form of w and must be the FIRST source of the multiply for ptxas to fold it).
__device__ __forceinline__ c2 cmul(c2 a, c2 w)
{
    float ax, ay, wx, wy;
    unpk(a, ax, ay);
    unpk(w, wx, wy);
    return fma2(bc(ax), w, mul2(pk(-wy, wx), bc(ay)));
}
// a * conj(w) = a.x (w.x, -w.y) + a.y (w.y, w.x)
__device__ __forceinline__ c2 cmulc(c2 a, c2 w)
{
    float ax, ay, wx, wy;
    unpk(a, ax, ay);
    unpk(w, wx, wy);
    return fma2(bc(ay), pk(wy, wx), mul2(pk(wx, -wy), bc(ax)));
}
__device__ __forceinline__ c2 csqr(c2 a) { return cmul(a, a); }
__device__ __forceinline__ c2 neg2(c2 a) { float x, y; unpk(a, x, y); return pk(-x, -y); }

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

// Butterfly lo = e + o w, hi = e - o w with w = e^{+2 pi i q / R}, 0 <= q < R/2 (compile-time
// after unrolling).  w = 1 or i: two FADD2; w = (+-1 + i)/sqrt 2: FADD2 + two FFMA2; general:
// lo = e + c (o.x, o.y) + s (-o.y, o.x) is two FFMA2 and hi = 2 e - lo a third.
template <int R>
__device__ __forceinline__ void bfly(const c2 e, const c2 o, const int q, c2& lo, c2& hi)
{
    const int a = q * (32 / R);                 // angle index, 0..15
    float ox, oy;
    unpk(o, ox, oy);
    if (a == 0) {
        lo = add2(e, o); hi = sub2(e, o);
    } else if (a == 8) {                        // w = i
        lo = add2(e, pk(-oy, ox)); hi = add2(e, pk(oy, -ox));
    } else if (a == 4) {                        // w = (1 + i) c :  o w = c (ox - oy, ox + oy)
        const float c = cos32_table(4);
        const c2 d = add2(o, pk(-oy, ox));
        lo = fma2(d, bc(c), e); hi = fma2(d, bc(-c), e);
    } else if (a == 12) {                       // w = (-1 + i) c : o w = -c (ox + oy, oy - ox)
        const float c = cos32_table(4);
        const c2 d = add2(o, pk(oy, -ox));
        lo = fma2(d, bc(-c), e); hi = fma2(d, bc(c), e);
    } else {
        const float c = (a <= 8) ? cos32_table(a) : -cos32_table(16 - a);
        const float s = (a <= 8) ? cos32_table(8 - a) : cos32_table(a - 8);
        // o w = c (ox, oy) + s (-oy, ox): the constants enter as BROADCAST scalars (immediates), the swap / sign flip
        // of o is an operand modifier -- no (c, s) register pairs to assemble
        lo = fma2(pk(-oy, ox), bc(s), fma2(o, bc(c), e));
        hi = fma2(e, bc(2.0f), neg2(lo));
    }
}

// Radix-R inverse DFT in registers, natural order in and out, decimation in time.
// NZ: only inputs v[0..NZ) are non-zero (the rest are never read), which prunes the leaves.
template <int R, int NZ>
struct DftP {
    static __device__ __forceinline__ void run(c2 (&v)[R])
    {
        if constexpr (NZ <= 1) {
#pragma unroll
            for (int q = 1; q < R; ++q) v[q] = v[0];
        } else {
            constexpr int H = R / 2;
            constexpr int NZE = ((NZ + 1) / 2 < H) ? (NZ + 1) / 2 : H;
            constexpr int NZO = (NZ / 2 < H) ? NZ / 2 : H;
            c2 e[H], o[H];
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
    static __device__ __forceinline__ void run(c2 (&)[1]) {}
};

template <int R>
__device__ __forceinline__ void dft(c2 (&v)[R]) { DftP<R, R>::run(v); }

// e^{+2 pi i num/den} with den a power of two <= 2^24 and 0 <= num < den: the argument of
// sincospif is formed exactly (integers below 2^24 and a power-of-two scale).
__device__ __forceinline__ c2 expi_frac(int num, float two_over_den)
{
    float s, c;
    sincospif((float)num * two_over_den, &s, &c);
    return pk(c, s);
}

// x[r] *= base * g^r for r = 0..R-1 (r = 0 multiplies by base only when HAS_BASE).
// Powers are built as g^(8 hi) * (base g^lo): every factor is at most 6 roundings deep.
template <int R, bool HAS_BASE>
__device__ __forceinline__ void mul_powers(c2 (&x)[R], c2 g, c2 base)
{
    constexpr int LO = (R < 8) ? R : 8;
    c2 pl[LO];
    const c2 g2 = csqr(g);
    if constexpr (HAS_BASE) {
        pl[0] = base;
        pl[1] = cmul(base, g);
    } else {
        pl[0] = pk(1.0f, 0.0f);
        pl[1] = g;
    }
    if constexpr (LO > 2) {
        const c2 g4 = csqr(g2);
        pl[2] = HAS_BASE ? cmul(pl[0], g2) : g2;
        pl[3] = cmul(pl[1], g2);
        if constexpr (LO > 4) {
            pl[4] = HAS_BASE ? cmul(pl[0], g4) : g4;
            pl[5] = cmul(pl[1], g4);
            pl[6] = cmul(pl[2], g4);
            pl[7] = cmul(pl[3], g4);
        }
        if constexpr (R > 8) {
            const c2 g8 = csqr(g4);
            c2 ph = g8;
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

// x[r] *= g^(r - R/2) for r = 0..R-1, R = 16 or 32: the twiddles x[r] g^r up to the factor g^(R/2)
// that is common to all R values.  Where only |DFT(x)|^2 matters (pass 2's arg-max epilogue) that
// unit-modulus factor can be left out, and the caller restores it for the few samples whose
// phase is reported.  g^k and its conjugate serve r = R/2 + k and R/2 - k, so R/2 - 1 products
// build the powers (against R - 2 in mul_powers) and R - 1 apply them.
template <int R>
__device__ __forceinline__ void mul_powers_centered(c2 (&x)[R], const c2 g)
{
    static_assert(R == 16 || R == 32, "mul_powers_centered: R = 16 or 32");
    constexpr int H = R / 2;
    c2 pl[8];
    pl[1] = g;
    pl[2] = csqr(g);
    pl[3] = cmul(pl[2], g);
    pl[4] = csqr(pl[2]);
    pl[5] = cmul(pl[4], g);
    pl[6] = cmul(pl[4], pl[2]);
    pl[7] = cmul(pl[4], pl[3]);
#pragma unroll
    for (int k = 1; k < 8; ++k) {
        x[H + k] = cmul(x[H + k], pl[k]);
        x[H - k] = cmulc(x[H - k], pl[k]);
    }
    const c2 g8 = csqr(pl[4]);
    if constexpr (R == 16) {
        x[0] = cmulc(x[0], g8);
    } else {
        x[H + 8] = cmul(x[H + 8], g8);
        x[H - 8] = cmulc(x[H - 8], g8);
#pragma unroll
        for (int k = 9; k < 16; ++k) {
            const c2 pk_ = cmul(g8, pl[k - 8]);
            x[H + k] = cmul(x[H + k], pk_);
            x[H - k] = cmulc(x[H - k], pk_);
        }
        x[0] = cmulc(x[0], csqr(g8));
    }
}

}  // namespace cbmf
