// kernels.cuh -- sm_100a kernels of the matched-filter hot path.
//
//   N = N1 * N2.  Frequency bin k = N2*k1 + k2, output sample j = j1 + N1*j2.
//   pass 1 (p1_kernel): for a tile of C adjacent columns k2, generate q~[k] = w[k] e^{+i Psi(f_k)}
//       in registers (S3, S4), N1-point inverse FFT over k1 -> Y[j1][k2]            (S5, first half)
//   pass 2 (p2_kernel): for ROWS adjacent rows j1, multiply by W_N^{j1 k2}, N2-point inverse FFT
//       over k2 -> z[j1 + N1 j2] in registers, |z|^2, arg-max, threshold              (S5-S7)
//   Y (N complex floats per template in flight) is the only materialised intermediate.  It is
//   stored tile-major, Y[k2 / NC][j1][k2 % NC] with NC = the columns of one pass-1 tile, so that the
//   output of a pass-1 block for one template is ONE contiguous piece, written by a TMA bulk store
//   from shared memory; pass 2 gathers a row from NC-column segments with asynchronous 16-byte copies.
//
// Each per-pass FFT is a Stockham autosort FFT whose butterflies (radix 8/16/32) live in
// registers and whose digit exchanges go through shared memory.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>
#include "fft_regs.cuh"

namespace cbmf {

// ------------------------------------------------------------------ per-template constants (S2)
struct __align__(16) TemplCoef {
    // phase in cycles: Psi/(2 pi) = A0 + u (A1 + u (A2 + u (A3 + u^2 A5))) + AL ln k,  u = k^{-1/3};
    // 2PN (BASELINE.json configs[0]): A0 = -1/8, AL = 0;  2.5PN (cbmf_set_pn_order, NEXT-3): AL ln k + const
    double A1, A2, A3, A5;
    int k_lo, k_hi;              // inclusive band on the DFT grid; empty if k_hi < k_lo
    float sigma, inv_sigma;      // sqrt(P[k_hi]), 1/sigma (0 for an empty band)
    float thr2;                  // (threshold * sigma)^2 : |z|^2 > thr2  <=>  rho > threshold
    float A0;                    // constant term, reduced to [-1/2, 1/2) cycles
    double AL;                   // coefficient of ln k (0 at 2PN)
};
static_assert(sizeof(TemplCoef) == 64, "TemplCoef layout");

// Status word of a bank call: index of its first invalid template (template_setup_kernel, atomicMin) or this value.
// The pass kernels of the call read it first and return at once when a template is invalid, so the host need not
// wait for the check before it enqueues them.
constexpr long long NO_BAD_TEMPLATE = 0x7FFFFFFFFFFFFFFFLL;

struct PeakOut { float snr_max; int32_t idx_peak; float phase; float sigma; };
struct TrigOut { int32_t template_idx; int32_t sample_idx; float snr; float phase; };

// ------------------------------------------------------------------ FFT configurations
template <int L> struct Cfg;
#define CBMF_CFG(L_, E_, R1_, R2_, R3_, NT1_)                                            \
    template <> struct Cfg<L_> {                                                         \
        static constexpr int E = E_, R1 = R1_, R2 = R2_, R3 = R3_, T = L_ / E_;          \
        static constexpr int NT1 = NT1_, NT2 = (L_ == 1024 ? 128 : 256);                                      \
        static constexpr int C = NT1 / T, ROWS = NT2 / T;                                \
        static constexpr int PADDED = L_ + L_ / R1_;                                     \
        static_assert(R1_ * R2_ * R3_ == L_, "radices");                                 \
    };
CBMF_CFG(64, 8, 8, 8, 1, 256)
CBMF_CFG(128, 16, 16, 8, 1, 256)
CBMF_CFG(256, 16, 16, 16, 1, 256)
CBMF_CFG(512, 32, 32, 16, 1, 256)
CBMF_CFG(1024, 32, 32, 32, 1, 256)
CBMF_CFG(2048, 32, 32, 32, 2, 512)
CBMF_CFG(4096, 32, 32, 32, 4, 512)
#undef CBMF_CFG

__host__ __device__ constexpr int ilog2c(int x) { return x <= 1 ? 0 : 1 + ilog2c(x >> 1); }

// cp.async (LDGSTS) helpers: 16-byte global -> shared copies that bypass registers and L1.
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src) : "memory");
}
// The same with compile-time byte offsets on both addresses: one base register pair serves a whole unrolled
// sequence of copies ([reg + imm] addressing instead of a 64-bit add per copy).
template <int SMEM_OFF, long long GMEM_OFF>
__device__ __forceinline__ void cp_async16_off(const unsigned smem_base, const void* gmem_base)
{
    asm volatile("cp.async.cg.shared.global [%0+%2], [%1+%3], 16;\n" ::"r"(smem_base), "l"(gmem_base), "n"(SMEM_OFF), "n"(GMEM_OFF)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

// Bulk asynchronous copy shared -> global (TMA, SASS UBLKCP): one thread hands `bytes` contiguous
// bytes to the copy engine; no registers and no LSU store slots are involved.
__device__ __forceinline__ void bulk_store(void* gmem_dst, const void* smem_src, const unsigned bytes)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_src);
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n" ::"l"(gmem_dst), "r"(s), "r"(bytes)
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;\n" ::: "memory");
}
// The copy engine has finished READING shared memory for every bulk store of this thread.
__device__ __forceinline__ void bulk_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;\n" ::: "memory"); }
// Writes to shared memory by this thread become visible to the copy engine (async proxy).
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

struct NoHook { __device__ __forceinline__ void operator()() const {} };

// Row stride (in c2) of the step-2 twiddle table TW[k][r] = e^{2 pi i k r / (R1 R2)}, k < R1,
// r < R2: even (rows are read with 16-byte loads) and = 2 mod 32 words so that the few rows a
// warp touches fall on different banks.
template <int L> __host__ __device__ constexpr int twtab_stride() { return Cfg<L>::R2 + 2; }
template <int L> __host__ __device__ constexpr int twtab_elems() { return Cfg<L>::R1 * twtab_stride<L>(); }

// Fill the step-2 twiddle table of an L-point FFT (all threads of the block take part).
template <int L>
__device__ __forceinline__ void twtab_fill(c2* __restrict__ tw, const int tid, const int nthreads)
{
    using C = Cfg<L>;
    for (int e = tid; e < C::R1 * C::R2; e += nthreads) {
        const int k = e / C::R2, r = e % C::R2;
        tw[k * twtab_stride<L>() + r] = expi_frac((k * r) & (C::R1 * C::R2 - 1), 2.0f / (float)(C::R1 * C::R2));
    }
}

// Stockham steps 1..3 of one L-point inverse FFT distributed over T threads (thread index t),
// E values per thread.  On entry v[u*R1 + r] = x[t + T*u + (L/R1)*r]; on exit
// v[u*RL + q] = X[t + T*u + (L/RL)*q] (RL = last radix).  sm points at this FFT's shared
// memory (element stride SS), padded by one element every R1.  NZ1: only r < NZ1 is non-zero.
//
// ROWTW (pass 2): the FFT is row j1 of the four-step decomposition and its input should have
// been multiplied by the inter-pass twiddle W_N^{j1 k2}, k2 = p0 + (L/R1) r, p0 = t + T u.
// The caller multiplies only by (W_N^{j1 L/R1})^r; the factor W_N^{j1 p0} is constant over
// the step-1 DFT, so it commutes with it and is folded here into the step-2 twiddles: the
// step-2 reader at position i + (L/R2) r' sees writer p0 = (i >> lg R1) + R3 r', i.e. an extra
// W_N^{j1 (i >> lg R1)} (W_N^{j1 R3})^{r'}.  n1 = N / L.
//
// tw (pass 1, may be null): the table of twtab_fill; the step-2 twiddles are then read from it
// instead of being built as powers (one multiply per element instead of two).
//
// after_last_read() is called once, after this thread's last read of the exchange buffer and
// before the arithmetic of the last step; pass 2 uses it to start the asynchronous copy of the
// next row into the same buffer (the hook must synchronise the group before it overwrites).
//
// SYNC: how the T threads of one FFT (or the threads sharing its exchange buffer) synchronise:
// the whole block, one warp, or a named barrier (bar_id, bar_threads) for a part of the block.
enum { SYNC_BLOCK = 0, SYNC_WARP = 1, SYNC_NAMED = 2 };
__device__ __forceinline__ void named_barrier(const int id, const int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
// CENTER (ROWTW, two-step FFTs): the step-2 twiddles are applied as g^(r - R2/2); every output of
// this thread then lacks the common factor g^(R2/2), with g = e^{2 pi i (k/(R1 R2) + j1/N)} and
// k = t mod R1 (see mul_powers_centered and fft_center_factor).
// Step 1 alone (radix R1, no twiddles, Ns = 1; output position i*R1 + q in the exchange buffer): callers that
// prune by the number of non-zero inputs instantiate only this part per NZ1 and share fft_core_tail.
template <int L, int NZ1, int SS>
__device__ __forceinline__ void fft_core_step1(c2 (&v)[Cfg<L>::E], const int t, c2* __restrict__ sm)
{
    using C = Cfg<L>;
    constexpr int E = C::E, T = C::T, R1 = C::R1;
    constexpr int LG_R1 = ilog2c(R1);
    auto pad = [](int pos) { return pos + (pos >> LG_R1); };
    constexpr int NB = E / R1;
#pragma unroll
    for (int u = 0; u < NB; ++u) {
        c2 x[R1];
#pragma unroll
        for (int r = 0; r < R1; ++r) x[r] = v[u * R1 + r];
        DftP<R1, NZ1>::run(x);
        const int i = t + T * u;
#pragma unroll
        for (int q = 0; q < R1; ++q) sm[(i * (R1 + 1) + q) * SS] = x[q];       // = pad(i R1 + q)
    }
}

template <int L, int SS, int SYNC, bool ROWTW, typename Hook = NoHook, bool CENTER = false>
__device__ __forceinline__ void fft_core_tail(c2 (&v)[Cfg<L>::E], const int t, c2* __restrict__ sm,
                                              const int j1 = 0, const int n1 = 1, Hook after_last_read = Hook(),
                                              const c2* __restrict__ tw = nullptr, const int bar_id = 0,
                                              const int bar_threads = 0, const c2* __restrict__ g_row = nullptr)
{
    using C = Cfg<L>;
    constexpr int E = C::E, T = C::T, R1 = C::R1, R2 = C::R2, R3 = C::R3;
    constexpr int LG_R1 = ilog2c(R1);
    auto pad = [](int pos) { return pos + (pos >> LG_R1); };
    auto sync = [&]() {
        if constexpr (SYNC == SYNC_WARP) __syncwarp();
        else if constexpr (SYNC == SYNC_NAMED) named_barrier(bar_id, bar_threads);
        else __syncthreads();
    };
    sync();
    // ---- step 2: radix R2, Ns = R1
    {
        constexpr int NB = E / R2, NS = R1;
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            // L/R2 is a multiple of R1, so pad(i + (L/R2) r) = pad(i) + r (L/R2)(1 + 1/R1): one base, constant offsets
            static_assert((L / R2) % R1 == 0, "step-2 stride");
            const int pi = pad(t + T * u);
#pragma unroll
            for (int r = 0; r < R2; ++r) v[u * R2 + r] = sm[(pi + r * ((L / R2) + (L / R2) / R1)) * SS];
        }
        if constexpr (R3 == 1) after_last_read();
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            c2 x[R2];
            const int i = t + T * u;
#pragma unroll
            for (int r = 0; r < R2; ++r) x[r] = v[u * R2 + r];
            const int k = i & (NS - 1);
            if constexpr (ROWTW) {
                // e^{2 pi i (k / (R1 R2) + j1 R3 / N)}: numerator over N = n1 L is an exact integer < N
                const float two_over_n = 2.0f / ((float)n1 * (float)L);
                // g_row (ROWTW, one step-2 DFT per thread): the caller carries g from row to row by a rotation
                const c2 g = (g_row != nullptr) ? *g_row : expi_frac(k * (n1 * R3) + j1 * R3, two_over_n);
                if constexpr (R3 > 1) {
                    mul_powers<R2, true>(x, g, expi_frac(j1 * (i >> LG_R1), two_over_n));
                } else if constexpr (CENTER) {
                    mul_powers_centered<R2>(x, g);
                } else {
                    mul_powers<R2, false>(x, g, pk(1.f, 0.f));
                }
            } else {
                if (tw != nullptr) {                 // uniform over the launch
                    const ulonglong2* __restrict__ row = reinterpret_cast<const ulonglong2*>(tw + k * twtab_stride<L>());
#pragma unroll
                    for (int r = 0; r < R2; r += 2) {
                        const ulonglong2 w2 = row[r / 2];
                        if (r > 0) x[r] = cmul(x[r], w2.x);
                        x[r + 1] = cmul(x[r + 1], w2.y);
                    }
                } else {
                    mul_powers<R2, false>(x, expi_frac(k, 2.0f / (float)(NS * R2)), pk(1.f, 0.f));
                }
            }
            dft<R2>(x);
#pragma unroll
            for (int q = 0; q < R2; ++q) v[u * R2 + q] = x[q];
        }
        if constexpr (R3 == 1) {
            return;
        } else {
            sync();   // all step-2 reads done before the buffer is overwritten
#pragma unroll
            for (int u = 0; u < NB; ++u) {
                const int i = t + T * u;
                const int k = i & (NS - 1);
                const int pb = pad((i >> LG_R1) * (NS * R2) + k);
#pragma unroll
                for (int q = 0; q < R2; ++q) sm[(pb + q * (NS + 1)) * SS] = v[u * R2 + q];      // NS = R1: pad(base + q R1) = pad(base) + q (R1 + 1)
            }
        }
    }
    if constexpr (R3 > 1) {
        sync();
        // ---- step 3: radix R3, Ns = R1*R2
        constexpr int NB = E / R3, NS = R1 * R2;
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            static_assert(R3 == 1 || (L / R3) % R1 == 0, "step-3 stride");
            const int pi = pad(t + T * u);
#pragma unroll
            for (int r = 0; r < R3; ++r) v[u * R3 + r] = sm[(pi + r * ((L / R3) + (L / R3) / R1)) * SS];
        }
        after_last_read();
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            c2 x[R3];
            const int i = t + T * u;
#pragma unroll
            for (int r = 0; r < R3; ++r) x[r] = v[u * R3 + r];
            const int k = i & (NS - 1);
            mul_powers<R3, false>(x, expi_frac(k, 2.0f / (float)L), pk(1.f, 0.f));
            dft<R3>(x);
#pragma unroll
            for (int q = 0; q < R3; ++q) v[u * R3 + q] = x[q];
        }
    }
}

template <int L, int NZ1, int SS, int SYNC, bool ROWTW, typename Hook = NoHook, bool CENTER = false>
__device__ __forceinline__ void fft_core(c2 (&v)[Cfg<L>::E], const int t, c2* __restrict__ sm,
                                         const int j1 = 0, const int n1 = 1, Hook after_last_read = Hook(),
                                         const c2* __restrict__ tw = nullptr, const int bar_id = 0,
                                         const int bar_threads = 0, const c2* __restrict__ g_row = nullptr)
{
    fft_core_step1<L, NZ1, SS>(v, t, sm);
    fft_core_tail<L, SS, SYNC, ROWTW, Hook, CENTER>(v, t, sm, j1, n1, after_last_read, tw, bar_id, bar_threads, g_row);
}

// The factor g^(R2/2) a CENTER transform leaves out of output element e (= u R2 + q) of thread t
// of row j1 (n1 = N / L).
template <int L>
__device__ __forceinline__ c2 fft_center_factor(const int t, const int e, const int j1, const int n1)
{
    using C = Cfg<L>;
    constexpr int R1 = C::R1, R2 = C::R2, T = C::T;
    const int k = (t + T * (e / R2)) & (R1 - 1);
    const long long num = ((long long)k * n1 + j1) * (R2 / 2);           // over N = n1 L
    const int n_total = n1 * L;
    return expi_frac((int)(num & (long long)(n_total - 1)), 2.0f / (float)n_total);
}

// ------------------------------------------------------------------ S3: SPA phasor
// e^{+i Psi_T(f_k)} for bin k >= 1 ("x form" in cycles).  The phase
// reaches 1e4 cycles, so the polynomial and the reduction to [-1/2, 1/2] cycles run in fp64
// (the FP64 pipe is otherwise idle); the fraction is then exact to 2^-32 cycles.
// u = k^{-1/3} in double comes from the template-independent table built by cbmf_create
// (rcbrt_table_kernel) or from the series of spa_correlate.  The reduced angle lies in [-pi, pi),
// where the SFU sine/cosine (MUFU.SIN/COS) have absolute error <= 2^-21.4 (CUDA math API,
// __sinf): a template mismatch of order 1e-13, against the 1e-6 bound of tests/parity.py.
struct SpaCoef { double A1, A2, A3, A5, AL; float A0; };
__device__ __forceinline__ SpaCoef spa_coef(const TemplCoef* __restrict__ tc)
{
    SpaCoef s;
    s.A1 = tc->A1; s.A2 = tc->A2; s.A3 = tc->A3; s.A5 = tc->A5; s.AL = tc->AL; s.A0 = tc->A0;
    return s;
}

// lnk: the table ln k of lnk_table_kernel (read only where AL != 0, i.e. at 2.5PN; may be null at 2PN)
__device__ __forceinline__ c2 spa_phasor_u(const double u, const int k, const SpaCoef& a, const double* __restrict__ lnk)
{
    double ph = fma(u * u, a.A5, a.A3);
    ph = fma(ph, u, a.A2);
    ph = fma(ph, u, a.A1);
    ph = fma(ph, u, (double)a.A0);
    if (a.AL != 0.0) ph = fma(a.AL, __ldg(lnk + k), ph);          // 2.5PN only (uniform over a template)
    // |ph| < 2^19 cycles: in ph + 1.5 * 2^20 the unit of the last place is 2^-32, so the low word of the
    // sum is the phase modulo one cycle as a 32-bit two's-complement fraction (one DADD, no conversion unit)
    const int frac = __double2loint(__dadd_rn(ph, 1572864.0));
    const float ang = (float)frac * (6.28318530717958647692f / 4294967296.0f);
    return pk(__cosf(ang), __sinf(ang));
}

// (double)f for a finite float |f| < 2^100 that is normal or zero, with integer instructions instead of
// the conversion unit (zero maps to 2^-127 ~ 5.9e-39, which the caller adds to a number of order 1e-2).
__device__ __forceinline__ double widen_f32(const float f)
{
    const unsigned b = __float_as_uint(f);
    const unsigned hi = (((b & 0x7FFFFFFFu) >> 3) + 0x38000000u) | (b & 0x80000000u);
    return __hiloint2double((int)hi, (int)(b << 29));
}

// u[k] = k^{-1/3} in double (k >= 1; u[0] = 0), one Newton step on the library cube root.
// lnk[k] = ln k in double (k >= 1; lnk[0] = 0): the 2.5PN phase term (cbmf_set_pn_order).
__global__ void lnk_table_kernel(double* __restrict__ lnk, int n_half)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n_half) lnk[k] = k > 0 ? log((double)k) : 0.0;
}

__global__ void rcbrt_table_kernel(double* __restrict__ u, int n_half)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_half) return;
    double r = 0.0;
    if (k > 0) {
        const double kd = (double)k;
        r = 1.0 / cbrt(kd);
        r = fma(r * fma(-kd * r, r * r, 1.0), 1.0 / 3.0, r);
    }
    u[k] = r;
}

// Position of Y[j1][k2] in the tile-major inter-pass buffer of one template.
template <int L1, int NC>
__device__ __forceinline__ size_t y_index(const int j1, const int k2)
{
    return ((size_t)(k2 / NC) * L1 + j1) * NC + (k2 % NC);
}

// S3 + S4 for the E/2 possibly non-zero inputs of one thread's column FFT:
// v[u R1 + r] = w[k] e^{+i Psi(f_k)}, k = (t + T u + (L/R1) r) L2 + k2, inside [k_lo, k_hi], else 0.
// The bins are taken four at a time: a group no lane of the warp needs is skipped (uniform
// branch), and inside a group the four phase chains (fp64 Horner, range reduction, SFU sine
// and cosine) are independent and branch-free, so their latencies overlap.
//   wt: this thread's column of w, row k1 at wt[k1 * WS];  ut: its column of k^{-1/3}, row k1 at
//   ut[k1 * US] (shared-memory tiles, or the global table with US = L2).
//   SERIES: k^{-1/3} is not loaded per bin but expanded about the first column of the tile,
//   k = kb + c with kb = k1 L2 + (first k2 of the tile):  k^{-1/3} = kb^{-1/3} (1 + d)^{-1/3},
//   d = c / kb,  (1 + d)^{-1/3} = 1 - d/3 + 2 d^2/9 - 14 d^3/81 + O(d^4).  ub[k1] = kb^{-1/3} (double)
//   and inv[k1] = 1/kb (float) sit in shared memory, cf = (float)c; the correction is below 1e-3 and
//   is evaluated in fp32 (absolute error ~1e-11), the caller guarantees d <= 2e-3 on every in-band
//   row (d^4 term < 3e-12).  This replaces a scattered 8-byte L2 load per bin, whose latency set the
//   length of the generator phase, by two shared-memory loads shared by the columns of a row.
template <int L, int L2, bool SERIES = false>
__device__ __forceinline__ void spa_correlate(c2 (&v)[Cfg<L>::E], const int t, const int k2,
                                              const c2* __restrict__ wt, const int WS,
                                              const double* __restrict__ ut, const int US,
                                              const int k_lo, const int k_hi, const SpaCoef& sc,
                                              const double* __restrict__ lnk,
                                              const double* __restrict__ ub = nullptr,
                                              const float* __restrict__ inv = nullptr, const float cf = 0.f)
{
    using C = Cfg<L>;
    constexpr int E = C::E, T = C::T, R1 = C::R1, NZ1 = R1 / 2;
    constexpr int G = (NZ1 < 4) ? NZ1 : 4;
#pragma unroll
    for (int u = 0; u < E / R1; ++u) {
#pragma unroll
        for (int rg = 0; rg < NZ1; rg += G) {
            const int k1a = t + T * u + (L / R1) * rg;
            const int ka = k1a * L2 + k2, kb = ka + (G - 1) * (L / R1) * L2;
            if (__any_sync(0xFFFFFFFFu, kb >= k_lo && ka <= k_hi)) {
#pragma unroll
                for (int j = 0; j < G; ++j) {
                    const int k1 = k1a + (L / R1) * j;
                    const int k = k1 * L2 + k2;
                    double uk;
                    if constexpr (SERIES) {
                        const float d = cf * inv[k1];
                        const float p = d * fmaf(d, fmaf(d, -14.0f / 81.0f, 2.0f / 9.0f), -1.0f / 3.0f);
                        const double b0 = ub[k1];
                        uk = fma(b0, widen_f32(p), b0);
                    } else {
                        uk = ut[(size_t)k1 * US];
                    }
                    const c2 ph = spa_phasor_u(uk, k, sc, lnk);
                    const c2 wv = (k >= k_lo && k <= k_hi) ? wt[k1 * WS] : czero();
                    v[u * R1 + rg + j] = cmul(ph, wv);
                }
            } else {
#pragma unroll
                for (int j = 0; j < G; ++j) v[u * R1 + rg + j] = czero();
            }
        }
#pragma unroll
        for (int r = NZ1; r < R1; ++r) v[u * R1 + r] = czero();
    }
}

// ------------------------------------------------------------------ S3 by rows (pass 1, two-step column FFTs)
// The NC columns of a pass-1 tile are consecutive bins k = kb + c of one row k1 (kb = k1 L2 + first column of the
// tile), so the phase in cycles, phi(k) = Psi_T(f_k) / 2 pi = -1/8 + A1 u + A2 u^2 + A3 u^3 + A5 u^5 with
// u = k^{-1/3}, is expanded about kb (D = d/dk, Du = -u^4 / 3):
//     phi(kb + c) = phi0 + c D phi + c^2 D2 phi / 2 + c^3 D3 phi / 6 + O(c^4 D4 phi),
//     D  phi = -(u^4 / 3)    (A1 +  2 A2 u +   3 A3 u^2 +   5 A5 u^4)
//     D2 phi =  (u^7 / 9)    (4 A1 + 10 A2 u +  18 A3 u^2 +  40 A5 u^4)
//     D3 phi = -(u^10 / 27) (28 A1 + 80 A2 u + 162 A3 u^2 + 440 A5 u^4)
// and evaluated ONCE per (template, row) instead of once per bin.  phi0 and D phi (up to 1e4 and a few cycles) are
// taken in fp64 and reduced modulo one cycle to 32-bit fixed point (units of 2^-32 cycle, the low word of
// x + 1.5 * 2^20 as in spa_phasor_u); D2 phi / 2 and D3 phi / 6 are below 1e-2 and 1e-7 cycles and are taken in
// fp32.  A bin then costs three wrapping integer multiply-adds (the reduction modulo one cycle is free), one
// conversion and the SFU sine / cosine.  The caller guarantees c / kb <= 2e-3 on every in-band row
// (p1_series_ok), where the neglected quartic term is below 3.2 (c/kb)^4 phi < 1e-6 cycle for phi < 1e4 cycles.
struct __align__(16) RowCoef { unsigned p0, p1; int p2, p3; };

__device__ __forceinline__ RowCoef spa_row_coef(const double u, const int kb, const SpaCoef& a, const double* __restrict__ lnk)
{
    const double A1 = a.A1, A2 = a.A2, A3 = a.A3, A5 = a.A5;
    const double u2 = u * u;
    double ph = fma(u2, A5, A3);
    ph = fma(ph, u, A2);
    ph = fma(ph, u, A1);
    ph = fma(ph, u, (double)a.A0);
    double q1 = fma(u2, 5.0 * A5, 3.0 * A3);
    q1 = fma(q1, u, 2.0 * A2);
    q1 = fma(q1, u, A1);
    double d1 = (-1.0 / 3.0) * (u2 * u2) * q1;
    const float uf = (float)u, uf2 = uf * uf, uf3 = uf2 * uf;
    const float a1 = (float)A1, a2 = (float)A2, a3 = (float)A3, a5 = (float)A5;
    float q2 = fmaf(uf2, 40.f * a5, 18.f * a3);
    q2 = fmaf(q2, uf, 10.f * a2);
    q2 = fmaf(q2, uf, 4.f * a1);
    float q3 = fmaf(uf2, 440.f * a5, 162.f * a3);
    q3 = fmaf(q3, uf, 80.f * a2);
    q3 = fmaf(q3, uf, 28.f * a1);
    const float uf7 = uf3 * uf3 * uf;
    float d2 = (4294967296.0f / 18.0f) * (uf7 * q2);             // D2 phi / 2 in units of 2^-32 cycle
    float d3 = (-4294967296.0f / 162.0f) * ((uf7 * uf3) * q3);   // D3 phi / 6
    if (a.AL != 0.0) {
        // 2.5PN: + AL ln k, with D = AL / k, D2 / 2 = -AL / (2 k^2), D3 / 6 = AL / (3 k^3)  (k^-1 = u^3)
        const double ik = u * u2;
        ph = fma(a.AL, __ldg(lnk + kb), ph);
        d1 = fma(a.AL, ik, d1);
        const float alf = (float)a.AL, ikf = (float)ik;
        d2 = fmaf(-0.5f * 4294967296.0f * alf, ikf * ikf, d2);
        d3 = fmaf((4294967296.0f / 3.0f) * alf, ikf * ikf * ikf, d3);
    }
    RowCoef r;
    r.p0 = (unsigned)__double2loint(__dadd_rn(ph, 1572864.0));
    r.p1 = (unsigned)__double2loint(__dadd_rn(d1, 1572864.0));
    r.p2 = __float2int_rn(d2);
    r.p3 = __float2int_rn(d3);
    return r;
}

// S3 + S4 from row records: v[r] = w[k] e^{+i Psi(f_k)}, k = (t + T r) L2 + k2, for r < NZ (the DFT that follows
// reads no other input); zero outside [k_lo, k_hi].  (c1, c2_, c3) = (c, c^2, c^3) of this thread's column c.
// Row record k1 sits at rc_lo[k1] for k1 < RS and at rc_hi[k1 - RS] above (RS a multiple of T: the choice is made at
// compile time for every r).
template <int L, int L2, int NZ, int RS>
__device__ __forceinline__ void spa_generate_rows(c2 (&v)[Cfg<L>::E], const int t, const int k2,
                                                  const c2* __restrict__ wt, const int WS,
                                                  const RowCoef* __restrict__ rc_lo, const RowCoef* __restrict__ rc_hi,
                                                  const int k_lo, const int k_hi,
                                                  const int c1, const int c2_, const int c3)
{
    using C = Cfg<L>;
    constexpr int T = C::T, R1 = C::R1;
    static_assert(C::E == R1, "one step-1 DFT per thread");
    static_assert(RS % T == 0, "row-record split on a multiple of T");
#pragma unroll
    for (int r = 0; r < NZ; ++r) {
        const int k1 = t + T * r;
        const int k = k1 * L2 + k2;
        const uint4 q = *reinterpret_cast<const uint4*>((T * r < RS) ? rc_lo + k1 : rc_hi + (k1 - RS));
        const unsigned ph = q.x + (unsigned)c1 * q.y + (unsigned)c2_ * q.z + (unsigned)c3 * q.w;
        const float ang = (float)(int)ph * (6.28318530717958647692f / 4294967296.0f);
        const c2 wv = (k >= k_lo && k <= k_hi) ? wt[k1 * WS] : czero();
        v[r] = cmul(pk(__cosf(ang), __sinf(ang)), wv);
    }
#pragma unroll
    for (int r = NZ; r < R1; ++r) v[r] = czero();
}

// ------------------------------------------------------------------ pass 1
// LOAD_GEN_DUMP (diagnostic): the generator of LOAD_GEN, bit for bit, but the generated inputs q~[k] are written to
// Y[b][k] in natural order and no FFT is run -- cbmf_debug_template reads the PRODUCT generator through it.
enum { LOAD_GEN = 0, LOAD_CPLX = 1, LOAD_REAL = 2, LOAD_GEN_DUMP = 3 };

struct P1Args {
    const c2* __restrict__ w;              // [N/2] weighted data spectrum (LOAD_GEN)
    const double* __restrict__ u;          // [N/2] k^{-1/3} (LOAD_GEN)
    const double* __restrict__ lnk;        // [N/2] ln k (LOAD_GEN at 2.5PN, else null)
    const TemplCoef* __restrict__ coef;    // [batch] (LOAD_GEN)
    const c2* __restrict__ in_c;           // [batch][N] (LOAD_CPLX)
    const float* __restrict__ in_r;        // [batch][N] (LOAD_REAL)
    c2* __restrict__ Y;                    // [batch][N], Y[j1*N2 + k2]
    int* err_flag;                         // set to 1 on a non-finite real input sample
    const long long* bad;                  // LOAD_GEN: *bad != NO_BAD_TEMPLATE (an invalid template in the bank): do nothing
    int batch;                             // templates (or vectors) in this launch
    int use_series;                        // LOAD_GEN: k^{-1/3} by the series of spa_correlate (host checks its range)
};

// The step-2 twiddle table is used where the FFT has two steps (L <= 1024).
template <int L> __host__ __device__ constexpr bool p1_use_twtab() { return Cfg<L>::R3 == 1; }

// The generator by rows (spa_generate_rows) serves the two-step column FFTs; the 2048- / 4096-point ones have no
// shared memory left for its tables and keep the per-bin series (spa_correlate).
template <int L> __host__ __device__ constexpr bool p1_by_rows() { return Cfg<L>::R3 == 1; }
// Row records k1 < p1_rc_split live in their own array, the others in the (L/R1) NC elements the padded exchange
// buffer has beyond the unpadded output tile.  At L = 1024 that keeps a block at 112.5 KiB, so that TWO blocks fit
// one SM (measured: 2 KiB more costs 16 % of the bank throughput).
template <int L> __host__ __device__ constexpr int p1_rc_split()
{
    constexpr int tail_rows = (Cfg<L>::PADDED - L) * Cfg<L>::C * (int)sizeof(c2) / 16;       // 16 = sizeof(RowCoef)
    constexpr int want = (L >= 1024) ? L / 2 - tail_rows : L / 2;
    return (want / Cfg<L>::T) * Cfg<L>::T + ((want % Cfg<L>::T) ? Cfg<L>::T : 0);
}

// Shared memory of one pass-1 block: the exchange buffer of NC column FFTs, the step-2 twiddle
// table and, for LOAD_GEN, the tile w[k1][k2 in tile], k1 < N1/2 (the upper half of the
// spectrum is zero), staged once per block and reused by every template the block works through.
template <int L1, int MODE_>
__host__ __device__ constexpr size_t p1_smem_bytes()
{
    using C = Cfg<L1>;
    constexpr int MODE = (MODE_ == LOAD_GEN_DUMP) ? LOAD_GEN : MODE_;
    return sizeof(c2) * ((size_t)C::PADDED * C::C + (p1_use_twtab<L1>() ? (size_t)twtab_elems<L1>() : 0) +
                         (MODE == LOAD_GEN ? (size_t)(L1 / 2) * C::C : 0)) +
           (MODE == LOAD_GEN ? (p1_by_rows<L1>() ? sizeof(RowCoef) * (size_t)p1_rc_split<L1>()                     // rc_lo
                                                 : (sizeof(double) + sizeof(float)) * (size_t)(L1 / 2))            // ub, inv
                             : 0);
}

// One pass-1 block = one tile of NC adjacent columns k2.  For every template slot b of the
// launch with b = blockIdx.y (mod gridDim.y): N1 = L1-point inverse FFT over k1 of
// x[k1*L2 + k2] -> Y[b][j1*L2 + k2].
template <int L1, int L2, int MODE_>
__global__ void __launch_bounds__(Cfg<L1>::NT1, (Cfg<L1>::NT1 <= 128 ? 4 : (Cfg<L1>::NT1 <= 256 ? 2 : 1))) p1_kernel(const P1Args a)
{
    extern __shared__ __align__(16) c2 smem[];
    using C = Cfg<L1>;
    constexpr int MODE = (MODE_ == LOAD_GEN_DUMP) ? LOAD_GEN : MODE_;
    constexpr bool DUMP = (MODE_ == LOAD_GEN_DUMP);
    constexpr int E = C::E, T = C::T, R1 = C::R1, NC = C::C, NT = C::NT1;
    constexpr int RL = (C::R3 > 1) ? C::R3 : C::R2;
    constexpr int NZ1 = (MODE == LOAD_GEN) ? R1 / 2 : R1;    // bins k >= N/2 are zero
    constexpr size_t n_total = (size_t)L1 * L2;
    constexpr bool TWTAB = p1_use_twtab<L1>();
    constexpr bool BYROWS = (MODE == LOAD_GEN) && p1_by_rows<L1>();
    constexpr int RS = p1_rc_split<L1>();                  // row records k1 < RS: own array; the rest: exchange-buffer tail

    if constexpr (MODE == LOAD_GEN) {
        if (a.bad != nullptr && __ldg(a.bad) != NO_BAD_TEMPLATE) return;               // uniform over the grid
    }
    const int tile = blockIdx.x;
    const int c = threadIdx.x % NC, t = threadIdx.x / NC;
    const int k2 = tile * NC + c;
    c2* __restrict__ tw = smem + (size_t)C::PADDED * NC;                               // [R1][R2 + 2]
    c2* __restrict__ wt = tw + (TWTAB ? twtab_elems<L1>() : 0);                          // [L1/2][NC]

    if constexpr (MODE == LOAD_GEN) {
        // stage the w tile: rows of NC complex = NC/2 chunks of 16 bytes
        constexpr int CPR = NC / 2, NCHUNK = (L1 / 2) * CPR;
        for (int ci = threadIdx.x; ci < NCHUNK; ci += NT) {
            const int row = ci / CPR, part = ci % CPR;
            cp_async16(wt + row * NC + 2 * part, a.w + ((size_t)row * L2 + tile * NC + 2 * part));
        }
        cp_async_commit();
    }
    if constexpr (TWTAB) twtab_fill<L1>(tw, threadIdx.x, NT);
    if constexpr (MODE != LOAD_GEN) __syncthreads();

    // ---- generator state
    // by rows (two-step FFTs): one RowCoef per row k1 < L1/2 of the CURRENT template -- rows below RS in their own
    // array after the w tile, the others in the tail of the exchange buffer that the unpadded output tile leaves
    // free (so that two pass-1 blocks still fit one SM); every thread keeps kb^{-1/3} of the RPT rows it fills.
    // per-bin series (three-step FFTs): tables kb^{-1/3} (double) and 1/kb of the first column, every row.
    RowCoef* __restrict__ rc_lo = reinterpret_cast<RowCoef*>(wt + (size_t)(L1 / 2) * NC);              // [RS]
    RowCoef* __restrict__ rc_hi = reinterpret_cast<RowCoef*>(smem + (size_t)L1 * NC);                   // [L1/2 - RS]
    double* __restrict__ ub = reinterpret_cast<double*>(wt + (size_t)(L1 / 2) * NC);                    // (!BYROWS)
    float* __restrict__ inv = reinterpret_cast<float*>(ub + L1 / 2);
    // Row records are WARP-LOCAL: a warp holds T_W = 32 / NC values of t and needs the rows k1 = t + T r, r < R1/2, of
    // exactly those; its 32 lanes fill them (RPT = T_W (R1/2) / 32 rows each: lane (t, c) takes r = c + NC i, so that
    // the rows of one i are the NC lowest ones still open and a band that ends below them skips that i for the whole
    // warp), so a __syncwarp orders fill and use and no block barrier is involved.  kb^{-1/3} of a lane's rows stays
    // in registers.
    static_assert(!BYROWS || (NC <= 32 && ((R1 / 2) % NC == 0 || NC % (R1 / 2) == 0)), "rows of a warp divide among its lanes");
    constexpr int RPT_W = ((R1 / 2) / NC > 1) ? (R1 / 2) / NC : 1;      // lanes c >= R1/2 of a wide tile stay idle
    double u_mine[RPT_W];
    if constexpr (MODE == LOAD_GEN) {
        if constexpr (BYROWS) {
#pragma unroll
            for (int i = 0; i < RPT_W; ++i) {
                const int k1 = t + T * (c + NC * i);
                u_mine[i] = (c + NC * i < R1 / 2) ? __ldg(a.u + (k1 * L2 + tile * NC)) : 0.0;
            }
        } else {
            for (int k1 = threadIdx.x; k1 < L1 / 2; k1 += NT) {
                const int kb = k1 * L2 + tile * NC;
                ub[k1] = __ldg(a.u + kb);
                inv[k1] = kb > 0 ? (float)(1.0 / (double)kb) : 0.f;
            }
        }
    }
    // row records of one template: those rows of this warp that touch the template's band
    auto fill_rows = [&](const TemplCoef* __restrict__ tn) {
        const int k_lo = tn->k_lo, k_hi = tn->k_hi;
        const SpaCoef sc = spa_coef(tn);
#pragma unroll
        for (int i = 0; i < RPT_W; ++i) {
            const int k1 = t + T * (c + NC * i);
            const int kb = k1 * L2 + tile * NC;
            if (c + NC * i < R1 / 2 && kb + NC - 1 >= k_lo && kb <= k_hi) {
                const RowCoef r = spa_row_coef(u_mine[i], kb, sc, a.lnk);
                if (k1 < RS) rc_lo[k1] = r; else rc_hi[k1 - RS] = r;
            }
        }
        __syncwarp();
    };

    // per-template constants travel through a two-entry shared buffer, fetched one template ahead
    __shared__ __align__(16) TemplCoef s_coef[2];
    const int G = gridDim.y;
    auto fetch_coef = [&](const int slot, const int bb) {
        if (threadIdx.x < 4 && bb < a.batch)
            cp_async16(reinterpret_cast<char*>(&s_coef[slot]) + 16 * threadIdx.x,
                       reinterpret_cast<const char*>(a.coef + bb) + 16 * threadIdx.x);
    };
    const bool by_rows = BYROWS && a.use_series;          // uniform over the launch
    if constexpr (MODE == LOAD_GEN) {
        fetch_coef(0, blockIdx.y);
        cp_async_commit();
        cp_async_wait_all();
        __syncthreads();
    }

    int cur = 0;
    for (int b = blockIdx.y; b < a.batch; b += G, cur ^= 1) {
        c2 v[E];
        bool step1_done = false;
        if constexpr (MODE == LOAD_GEN) {
            fetch_coef(cur ^ 1, b + G);
            cp_async_commit();
            const TemplCoef* tc = &s_coef[cur];
            if constexpr (BYROWS) {
                if (by_rows) {
                    // this template's row records (the previous ones were last read by this warp in the previous
                    // iteration; the exchange-buffer tail is free between the step-2 reads and the step-1 writes);
                    // the copy engine drains the previous output tile meanwhile
                    fill_rows(tc);
                    const int k_lo = tc->k_lo, k_hi = tc->k_hi;
                    // inputs v[r] = x[t + T r] beyond the band are zero: prune the step-1 DFT to NZ of them (uniform)
                    const int nz = (k_hi < 0) ? 0 : ((k_hi / L2) / T + 1);
                    auto run = [&](auto nz_tag) {
                        constexpr int NZ = decltype(nz_tag)::value;
                        spa_generate_rows<L1, L2, NZ, RS>(v, t, k2, wt + c, NC, rc_lo, rc_hi, k_lo, k_hi, c, c * c, c * c * c);
                        if constexpr (!DUMP) {
                            // the copy engine may still be reading the previous output tile out of the exchange buffer
                            if (threadIdx.x == 0) bulk_store_wait_read();
                            __syncthreads();
                            fft_core_step1<L1, NZ, NC>(v, t, smem + c);
                        }
                    };
                    if constexpr (R1 >= 32) {
                        switch (nz) {
                            case 0: case 1: case 2: run(std::integral_constant<int, 2>()); break;
                            case 3: run(std::integral_constant<int, 3>()); break;
                            case 4: run(std::integral_constant<int, 4>()); break;
                            case 5: run(std::integral_constant<int, 5>()); break;
                            case 6: run(std::integral_constant<int, 6>()); break;
                            case 7: run(std::integral_constant<int, 7>()); break;
                            case 8: run(std::integral_constant<int, 8>()); break;
                            case 9: run(std::integral_constant<int, 9>()); break;
                            case 10: run(std::integral_constant<int, 10>()); break;
                            case 11: run(std::integral_constant<int, 11>()); break;
                            case 12: run(std::integral_constant<int, 12>()); break;
                            case 13: run(std::integral_constant<int, 13>()); break;
                            case 14: run(std::integral_constant<int, 14>()); break;
                            case 15: run(std::integral_constant<int, 15>()); break;
                            default: run(std::integral_constant<int, 16>()); break;
                        }
                    } else if constexpr (R1 >= 16) {
                        if (nz <= 2) run(std::integral_constant<int, 2>());
                        else if (nz <= 4) run(std::integral_constant<int, 4>());
                        else if (nz <= 6) run(std::integral_constant<int, 6>());
                        else run(std::integral_constant<int, 8>());
                    } else {
                        if (nz <= 2) run(std::integral_constant<int, 2>());
                        else run(std::integral_constant<int, R1 / 2>());
                    }
                    step1_done = true;
                }
            }
            if (!step1_done) {
                if constexpr (!BYROWS) {
                    if (a.use_series)
                        spa_correlate<L1, L2, true>(v, t, k2, wt + c, NC, nullptr, 0, tc->k_lo, tc->k_hi, spa_coef(tc), a.lnk, ub, inv,
                                                    (float)c);
                    else
                        spa_correlate<L1, L2>(v, t, k2, wt + c, NC, a.u + k2, L2, tc->k_lo, tc->k_hi, spa_coef(tc), a.lnk);
                } else {
                    spa_correlate<L1, L2>(v, t, k2, wt + c, NC, a.u + k2, L2, tc->k_lo, tc->k_hi, spa_coef(tc), a.lnk);
                }
            }
        } else {
#pragma unroll
            for (int u = 0; u < E / R1; ++u) {
#pragma unroll
                for (int r = 0; r < R1; ++r) {
                    const size_t k = (size_t)(t + T * u + (L1 / R1) * r) * L2 + k2;
                    if constexpr (MODE == LOAD_CPLX) {
                        v[u * R1 + r] = __ldg(a.in_c + (size_t)b * n_total + k);
                    } else {
                        const float x = __ldg(a.in_r + (size_t)b * n_total + k);
                        if (!isfinite(x)) *a.err_flag = 1;
                        v[u * R1 + r] = pk(x, 0.f);
                    }
                }
            }
        }

        if constexpr (DUMP) {
#pragma unroll
            for (int r = 0; r < R1; ++r)
                a.Y[(size_t)b * n_total + (size_t)(t + T * r) * L2 + k2] = v[r];
            cp_async_wait_all();
            __syncthreads();
            continue;
        }
        if (!step1_done) {
            // the copy engine may still be reading the previous template's output tile out of the exchange buffer
            if (threadIdx.x == 0) bulk_store_wait_read();
            __syncthreads();
            fft_core_step1<L1, NZ1, NC>(v, t, smem + c);
        }
        fft_core_tail<L1, NC, SYNC_BLOCK, false>(v, t, smem + c, 0, 1, NoHook(), TWTAB ? tw : nullptr);

        // Y[b][tile] (L1 rows of NC columns) is one contiguous block of the tile-major buffer: build it in
        // the exchange buffer, unpadded, and hand it to the copy engine in one piece.
        if constexpr (MODE == LOAD_GEN) cp_async_wait_all();   // the next template's constants have landed
        __syncthreads();                              // every step-2 read of the exchange buffer is done
        c2* __restrict__ ot = smem + (size_t)t * NC + c;
#pragma unroll
        for (int u = 0; u < E / RL; ++u) {
#pragma unroll
            for (int q = 0; q < RL; ++q)
                ot[(size_t)(T * u + (L1 / RL) * q) * NC] = v[u * RL + q];     // row j1 = t + T u + (L1/RL) q
        }
        fence_async_smem();
        __syncthreads();
        if (threadIdx.x == 0)
            bulk_store(a.Y + (size_t)b * n_total + (size_t)tile * L1 * NC, smem, (unsigned)(sizeof(c2) * L1 * NC));
    }
    if (threadIdx.x == 0) bulk_store_wait_read();     // shared memory must outlive the last copy
}

// ------------------------------------------------------------------ pass 2
enum { EPI_MAX = 0, EPI_STORE = 1, EPI_WSTORE = 2 };

struct P2Args {
    const c2* __restrict__ Y;              // [batch][N]
    // EPI_MAX
    const TemplCoef* __restrict__ coef;    // [batch]
    unsigned long long* best_key;          // [batch] running arg-max key, zero on entry, zero again on exit
    c2* cand;                              // [batch][N / E]  z at the candidate of (row j1, thread t)
    unsigned int* done_ctr;                // [batch], zero on entry, zero again on exit
    PeakOut* peaks;                        // [batch] (already offset to this sub-batch)
    TrigOut* trig;                         // bounded trigger list
    unsigned long long* trig_cursor;       // total found so far
    unsigned long long trig_cap;
    unsigned int* trig_count;              // [batch] triggers found per template (for a deterministic truncated list)
    int tmpl_base;                         // bank index of template 0 of this sub-batch
    int j_min;                             // MASK: samples j < j_min take no part in the peak or the trigger list
    const long long* bad;                  // EPI_MAX: *bad != NO_BAD_TEMPLATE: do nothing
    // EPI_STORE
    c2* __restrict__ z_out;                // [batch][N], natural order
    // EPI_WSTORE (load_segment): w[k] = conj(Z[k]) * wfac[k] for k < N/2
    c2* __restrict__ w_out;                // [N/2]
    const double* __restrict__ wfac;       // [N/2]
};

// (|z|^2 bits, ~j): the larger value wins and, among equal values, the smaller sample index,
// whatever the order of arrival (|z|^2 >= 0, so its bit pattern orders like the value).
__device__ __forceinline__ unsigned long long pack_key(float p, int j)
{
    return ((unsigned long long)__float_as_uint(p) << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned)j);
}

// Rows each thread group walks in the arg-max pass.
template <int L1, int L2>
__host__ __device__ constexpr int p2_rpw()
{
    constexpr int per8 = L1 / Cfg<L2>::ROWS / 8;
    return per8 >= 16 ? 16 : (per8 >= 1 ? per8 : 1);
}
template <int L2> __host__ __device__ constexpr int p2_row_stride()
{
    return Cfg<L2>::PADDED + (Cfg<L2>::T <= 32 ? Cfg<L2>::R1 : 0);      // exchange buffer + G table
}

// Start the asynchronous copy of row j1 of one template's Y (tile-major: segments of NC columns)
// into the row group's shared-memory buffer (unpadded, element k2 at sm[k2]); T threads take part.
template <int L1, int L2, int I>
struct P2Prefetch {
    // chunk I of a thread: columns k2 = 2 (t + T I), k2 + 1; consecutive chunks lie 2 T / NC tiles = 2 T L1 elements apart
    static __device__ __forceinline__ void run(const unsigned sm_t, const c2* __restrict__ src_t)
    {
        constexpr int T = Cfg<L2>::T, E = Cfg<L2>::E;
        if constexpr (I < E / 2) {
            cp_async16_off<(int)(sizeof(c2) * 2 * T * I), (long long)(sizeof(c2) * 2 * T * L1) * I>(sm_t, src_t);
            P2Prefetch<L1, L2, I + 1>::run(sm_t, src_t);
        }
    }
};
template <int L1, int L2>
__device__ __forceinline__ void p2_prefetch_row(c2* __restrict__ sm, const c2* __restrict__ yb, const int j1, const int t)
{
    constexpr int T = Cfg<L2>::T, E = Cfg<L2>::E, NC = Cfg<L1>::C;
    static_assert(NC % 2 == 0, "16-byte chunks must not straddle tiles");
    // the chunks of one thread are whole tiles apart and the largest offset fits the immediate field of the copy
    constexpr bool IMM = ((2 * T) % NC == 0) && ((long long)sizeof(c2) * 2 * T * L1 * (E / 2 - 1) < (1LL << 23));
    if constexpr (IMM) {
        P2Prefetch<L1, L2, 0>::run((unsigned)__cvta_generic_to_shared(sm + 2 * t), yb + y_index<L1, NC>(j1, 2 * t));
    } else {
#pragma unroll
        for (int i = 0; i < E / 2; ++i) {
            const int k2 = 2 * (t + T * i);
            cp_async16(sm + k2, yb + y_index<L1, NC>(j1, k2));
        }
    }
    cp_async_commit();
}

// Row-to-row twiddle state of one pass-2 thread (EPI_MAX, rows of 1024 points: one warp per row, one
// DFT per thread and step).  Both row-dependent twiddle seeds are pure phases that advance by a
// constant angle when the warp moves on by `stride` rows, so after the first row of an item (two
// sincospi per thread) they are carried by one complex multiply each instead of being recomputed:
//   G  = e^{2 pi i j1 t / (L1 R1)}        the lane's entry of the (W_N^{j1 L2/R1})^r table,  dG = e^{2 pi i stride t / (L1 R1)}
//   g  = e^{2 pi i (t n1 + j1) / N}       the step-2 twiddle seed of fft_core (k = t),       dg = e^{2 pi i stride / N}
// At most 16 rows follow one initialisation: the accumulated rounding is ~1e-6 of the phase.
template <int L1, int L2>
struct P2Tw {
    static constexpr bool ON = (Cfg<L2>::T == 32) && (Cfg<L2>::E == Cfg<L2>::R1) && (Cfg<L2>::E == Cfg<L2>::R2) &&
                               (Cfg<L2>::R3 == 1);
    c2 G, dG, g, dg;
    __device__ __forceinline__ void init(const int j1, const int stride, const int t)
    {
        if constexpr (ON) {
            constexpr int R1 = Cfg<L2>::R1;
            const float s1 = 2.0f / (float)(L1 * R1), sn = 2.0f / ((float)L1 * (float)L2);
            G = expi_frac((j1 * t) & (L1 * R1 - 1), s1);
            dG = expi_frac((stride * t) & (L1 * R1 - 1), s1);
            g = expi_frac(t * L1 + j1, sn);
            dg = expi_frac(stride, sn);
        }
    }
    __device__ __forceinline__ void advance()
    {
        if constexpr (ON) { G = cmul(G, dG); g = cmul(g, dg); }
    }
};

// Row j1 of template slot b: twiddle, N2 = L2-point inverse FFT over k2 -> z[j1 + L1 j2] in
// registers, then the epilogue of MODE.  Called by the T threads of one row group.  On entry the
// copy of the row into sm has been started by p2_prefetch_row; next_j1 (or -1) is the row of the
// same template (yb) whose copy is started as soon as the exchange buffer is free again.
template <int L1, int L2, int MODE, bool MASK = false>
__device__ __forceinline__ void p2_row(const P2Args& a, const int j1, const int b, const int t,
                                       c2* __restrict__ sm, const c2* __restrict__ yb, const int next_j1,
                                       P2Tw<L1, L2>& rtw)
{
    constexpr bool ROT = P2Tw<L1, L2>::ON && (MODE == EPI_MAX);
    using C = Cfg<L2>;
    constexpr int E = C::E, T = C::T, R1 = C::R1;
    constexpr int RL = (C::R3 > 1) ? C::R3 : C::R2;
    constexpr bool WSYNC = (T <= 32);
    constexpr int LG1 = ilog2c(L1);
    constexpr size_t n_total = (size_t)L1 * L2;
    auto gsync = []() { if constexpr (WSYNC) __syncwarp(); else __syncthreads(); };

    // the running maximum of this template, read early (S7): rows that cannot beat it skip the search
    unsigned best_bits = 0u;
    if constexpr (MODE == EPI_MAX) best_bits = (unsigned)(__ldcg(a.best_key + b) >> 32);

    // row j1 from the staging buffer; multiply by (W_N^{j1 L2/R1})^r (the rest of the inter-pass
    // twiddle is folded into the step-2 twiddles of fft_core)
    c2 v[E];
    cp_async_wait_all();
    gsync();
#pragma unroll
    for (int u = 0; u < E / R1; ++u)
#pragma unroll
        for (int r = 0; r < R1; ++r) v[u * R1 + r] = sm[t + T * u + (L2 / R1) * r];
    if constexpr (WSYNC) {
        // G[r] = e^{2 pi i j1 r / (L1 R1)}, r < R1: one sincospi per lane, broadcast through shared memory
        c2* __restrict__ G = sm + C::PADDED;
        if constexpr (ROT) {
            G[t] = rtw.G;
        } else {
            for (int r = t; r < R1; r += T) G[r] = expi_frac((j1 * r) & (L1 * R1 - 1), 2.0f / (float)(L1 * R1));
        }
        __syncwarp();
#pragma unroll
        for (int r = 2; r < R1; r += 2) {
            const ulonglong2 g = *reinterpret_cast<const ulonglong2*>(G + r);
#pragma unroll
            for (int u = 0; u < E / R1; ++u) {
                v[u * R1 + r] = cmul(v[u * R1 + r], g.x);
                v[u * R1 + r + 1] = cmul(v[u * R1 + r + 1], g.y);
            }
        }
        {
            const c2 g1 = G[1];
#pragma unroll
            for (int u = 0; u < E / R1; ++u) v[u * R1 + 1] = cmul(v[u * R1 + 1], g1);
        }
    } else {
        __syncthreads();                                              // staging reads done before the exchange writes
        const c2 g = expi_frac(j1, 2.0f / (float)(L1 * R1));          // W_N^{j1 L2/R1}
#pragma unroll
        for (int u = 0; u < E / R1; ++u) {
            c2 x[R1];
#pragma unroll
            for (int r = 0; r < R1; ++r) x[r] = v[u * R1 + r];
            mul_powers<R1, false>(x, g, pk(1.f, 0.f));
#pragma unroll
            for (int r = 0; r < R1; ++r) v[u * R1 + r] = x[r];
        }
    }

    auto start_next = [&]() {
        if (next_j1 >= 0) {                 // uniform over the row group
            gsync();                        // every thread of the group has read the exchange buffer
            p2_prefetch_row<L1, L2>(sm, yb, next_j1, t);
        }
    };
    // in the arg-max pass only |z|^2 is needed for almost every sample: leave the common factor out
    constexpr bool CENTER = (MODE == EPI_MAX) && (C::R3 == 1) && (C::R2 == 16 || C::R2 == 32);
    fft_core<L2, R1, 1, (WSYNC ? SYNC_WARP : SYNC_BLOCK), true, decltype(start_next), CENTER>(
        v, t, sm, j1, L1, start_next, nullptr, 0, 0, ROT ? &rtw.g : nullptr);
    if constexpr (ROT) rtw.advance();

    // v[u*RL + q] = z[j1 + L1 * j2],  j2 = t + T u + (L2/RL) q
    if constexpr (MODE == EPI_STORE || MODE == EPI_WSTORE) {
        // z[j1 + L1 j2]: a thread's outputs lie L1 samples apart, so direct stores would touch one 32-byte sector per
        // 8-byte value (four times the sector writes: 2.0 ms instead of 1.1 ms per 256 transforms at N = 2^20).  The
        // ROWS adjacent rows of the block are transposed through its shared memory instead (T[j2][row], one pad element
        // every PAD values of j2 against bank conflicts) and leave as runs of ROWS consecutive samples.
        constexpr int ROWS = C::ROWS, NT = C::NT2;
        constexpr int CAP = ROWS * p2_row_stride<L2>();
        constexpr int SPARE = CAP - L2 * ROWS;
        static_assert(SPARE > 0, "transposed store needs spare shared memory");
        constexpr int PAD_MIN = (L2 + SPARE - 1) / SPARE;
        constexpr int PAD = PAD_MIN <= 4 ? 4 : (PAD_MIN <= 8 ? 8 : (PAD_MIN <= 16 ? 16 : 32));
        static_assert(L2 * ROWS + L2 / PAD <= CAP, "transposed store fits the block's buffers");
        const int row = threadIdx.x / T;
        c2* __restrict__ tt = sm - row * p2_row_stride<L2>();
        __syncthreads();                                    // every row group has read its exchange buffer
#pragma unroll
        for (int u = 0; u < E / RL; ++u)
#pragma unroll
            for (int q = 0; q < RL; ++q) {
                const int j2 = t + T * u + (L2 / RL) * q;
                tt[j2 * ROWS + j2 / PAD + row] = v[u * RL + q];
            }
        __syncthreads();
        if constexpr (MODE == EPI_STORE) {
            c2* __restrict__ zb = a.z_out + (size_t)b * n_total + (j1 - row);
#pragma unroll 8
            for (int m = threadIdx.x; m < L2 * ROWS; m += NT) {
                const int j2 = m / ROWS, r = m % ROWS;
                zb[((size_t)j2 << LG1) + r] = tt[m + j2 / PAD];
            }
        } else {
            // load_segment: w[k] = conj(Z[k]) wfac[k] for k_lo <= k < N/2, zero below
            const int k_lo = a.coef->k_lo;
#pragma unroll 4
            for (int m = threadIdx.x; m < L2 * ROWS / 2; m += NT) {     // j2 < L2 / 2: k < N / 2
                const int j2 = m / ROWS, r = m % ROWS;
                const size_t k = ((size_t)j2 << LG1) + (size_t)(j1 - row + r);
                c2 o = czero();
                if ((long long)k >= k_lo) {
                    const c2 zv = tt[m + j2 / PAD];
                    const double f = a.wfac[k];
                    o = pk((float)(f * (double)re(zv)), (float)(-f * (double)im(zv)));
                }
                a.w_out[k] = o;
            }
        }
    } else {
        // ---- S6/S7: |z|^2, arg-max (lowest index on ties), threshold.
        // Fast path: the thread's maximum of |z|^2 against the template's running maximum (read at
        // the start of the row) and against the threshold.  A thread that may hold a new maximum
        // locates its sample, publishes (|z|^2, ~j) with one 64-bit atomicMax and, if it won,
        // leaves z in its own candidate slot (j1, t) for the block that finishes the template.
        const TemplCoef* tc = a.coef + b;
        const float thr2 = tc->thr2, inv_sigma = tc->inv_sigma;
        // MASK (segment streaming): sample j = j1 + L1 j2 counts only if j >= j_min, i.e. j2 >= j2_min on this row;
        // an excluded sample reads as -1, below every |z|^2 and every threshold
        const int j2_min = MASK ? max(0, (a.j_min - j1 + L1 - 1) >> LG1) : 0;
        auto pw = [&](int e) {
            float x, y;
            unpk(v[e], x, y);
            float p = fmaf(x, x, y * y);
            if constexpr (MASK) {
                if (t + T * (e / RL) + (L2 / RL) * (e % RL) < j2_min) p = -1.0f;
            }
            return p;
        };
        float m = pw(0);
#pragma unroll
        for (int e = 1; e < E; ++e) m = fmaxf(m, pw(e));
        const unsigned mbits = __float_as_uint(m);
        if (mbits >= best_bits && (!MASK || m >= 0.f)) {
            // only the lanes holding the group's largest value go on (usually one per warp)
            unsigned gm = mbits;
            if constexpr (WSYNC) gm = __reduce_max_sync(__activemask(), mbits);
            if (mbits == gm) {
                int best_e = 0;
                bool found = false;
#pragma unroll
                for (int q = 0; q < RL; ++q)        // j2 increases with (q, u): first maximum kept
#pragma unroll
                    for (int u = 0; u < E / RL; ++u) {
                        const int e = u * RL + q;
                        if (!found && pw(e) == m) { found = true; best_e = e; }
                    }
                const int j2 = t + T * (best_e / RL) + (L2 / RL) * (best_e % RL);
                const int j = (j2 << LG1) + j1;
                const unsigned long long key = pack_key(m, j);
                const unsigned long long old = atomicMax(a.best_key + b, key);
                if (old < key) {
                    c2 zb = v[0];
#pragma unroll
                    for (int e = 1; e < E; ++e)
                        if (e == best_e) zb = v[e];
                    if constexpr (CENTER) zb = cmul(zb, fft_center_factor<L2>(t, best_e, j1, L1));
                    __stcg(a.cand + (size_t)b * (n_total / E) + (size_t)j1 * T + t, zb);
                }
            }
        }
        if (m > thr2 && inv_sigma > 0.f) {
            // one slot range per thread: count, reserve, write (order inside the list is restored by the sort)
            unsigned n_mine = 0;
#pragma unroll
            for (int e = 0; e < E; ++e) n_mine += (pw(e) > thr2) ? 1u : 0u;
            unsigned long long slot = atomicAdd(a.trig_cursor, (unsigned long long)n_mine);
            atomicAdd(a.trig_count + b, n_mine);
#pragma unroll
            for (int q = 0; q < RL; ++q)
#pragma unroll
                for (int u = 0; u < E / RL; ++u) {
                    const int e = u * RL + q;
                    const float pe = pw(e);
                    if (pe > thr2) {
                        if (slot < a.trig_cap) {
                            const int j2 = t + T * u + (L2 / RL) * q;
                            TrigOut o;
                            o.template_idx = a.tmpl_base + b;
                            o.sample_idx = (j2 << LG1) + j1;
                            o.snr = sqrtf(pe) * inv_sigma;
                            c2 zt = v[e];
                            if constexpr (CENTER) zt = cmul(zt, fft_center_factor<L2>(t, e, j1, L1));
                            o.phase = atan2f(im(zt), re(zt));
                            a.trig[slot] = o;
                        }
                        ++slot;
                    }
                }
        }
    }
}

// Block-level end of the arg-max pass: the last of the n_items blocks of template slot b turns
// the template's key and the winner's candidate slot into the PeakOut record.
template <int L1, int L2>
__device__ __forceinline__ void p2_finish(const P2Args& a, const int b, const int n_items)
{
    using C = Cfg<L2>;
    constexpr int LG1 = ilog2c(L1);
    constexpr size_t n_total = (size_t)L1 * L2;
    __syncthreads();                                // every row of this block has published
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int prev = atomicAdd(a.done_ctr + b, 1u);
        if (prev == (unsigned)n_items - 1u) {
            __threadfence();
            const TemplCoef* tc = a.coef + b;
            const unsigned long long bk = __ldcg(a.best_key + b);
            PeakOut o;
            if (tc->k_hi < tc->k_lo) {              // empty band
                o.snr_max = 0.f; o.idx_peak = -1; o.phase = 0.f; o.sigma = 0.f;
            } else {
                const float p = __uint_as_float((unsigned)(bk >> 32));
                const int j = (int)(0xFFFFFFFFu - (unsigned)(bk & 0xFFFFFFFFu));
                const int j1 = j & (L1 - 1), tt = (j >> LG1) & (C::T - 1);
                const c2 z = __ldcg(a.cand + (size_t)b * (n_total / C::E) + (size_t)j1 * C::T + tt);
                o.snr_max = sqrtf(p) * tc->inv_sigma;
                o.idx_peak = j;
                o.phase = atan2f(im(z), re(z));
                o.sigma = tc->sigma;
            }
            a.peaks[b] = o;
            a.best_key[b] = 0ULL;                   // self-cleaning for the next launch
            a.done_ctr[b] = 0u;
        }
    }
}

// One item of pass 2: ROWS * RPW rows of template slot b.
template <int L1, int L2, int MODE, bool MASK = false>
__device__ __forceinline__ void p2_item(const P2Args& a, const int item, const int b, c2* __restrict__ smem)
{
    using C = Cfg<L2>;
    constexpr int T = C::T, ROWS = C::ROWS;
    constexpr int RPW = (MODE == EPI_MAX) ? p2_rpw<L1, L2>() : 1;
    constexpr size_t n_total = (size_t)L1 * L2;
    const int t = threadIdx.x % T, row = threadIdx.x / T;
    c2* sm = smem + row * p2_row_stride<L2>();
    const c2* __restrict__ yb = a.Y + (size_t)b * n_total;
    p2_prefetch_row<L1, L2>(sm, yb, (item * RPW) * ROWS + row, t);
    P2Tw<L1, L2> rtw;
    if constexpr (MODE == EPI_MAX) rtw.init((item * RPW) * ROWS + row, ROWS, t);
#pragma unroll 1
    for (int it = 0; it < RPW; ++it) {
        const int j1 = (item * RPW + it) * ROWS + row;
        p2_row<L1, L2, MODE, MASK>(a, j1, b, t, sm, yb, (it + 1 < RPW) ? j1 + ROWS : -1, rtw);
    }
    if constexpr (MODE == EPI_MAX) p2_finish<L1, L2>(a, b, L1 / (ROWS * RPW));
}

template <int L1, int L2, int MODE, bool MASK = false>
__global__ void __launch_bounds__(Cfg<L2>::NT2, 512 / Cfg<L2>::NT2) p2_kernel(const P2Args a)
{
    extern __shared__ __align__(16) c2 smem[];
    if constexpr (MODE == EPI_MAX) {
        if (a.bad != nullptr && __ldg(a.bad) != NO_BAD_TEMPLATE) return;               // uniform over the grid
    }
    // templates in reverse order: pass 1 wrote the last ones most recently, so part of their Y is still in the L2
    // when this launch starts (4 % fewer DRAM reads of a launch timed alone)
    p2_item<L1, L2, MODE, MASK>(a, blockIdx.x, gridDim.y - 1 - blockIdx.y, smem);
}

// ------------------------------------------------------------------ S0: PSD tables (fp64)
// wfac[k] = 4 df dt f_k^{-7/6} / S_n[k]; term[k] = 4 df f_k^{-7/3} / S_n[k]  (0 outside
// [k_lo, N/2) or where S_n = +inf).  err_flag = 1 if S_n <= 0 or NaN inside the band.
// prefix[k] = sum_{k' <= k} term[k'] is built by a three-launch scan: every block of
// SCAN_TILE bins writes its total (psd_terms_kernel), one block scans the totals
// (scan_block_sums_kernel), every block rescans its tile from its offset (prefix_tile_kernel).
constexpr int SCAN_THREADS = 256, SCAN_PER_THREAD = 4, SCAN_TILE = SCAN_THREADS * SCAN_PER_THREAD;

// Exclusive scan of one value per thread over a block of SCAN_THREADS threads; *total = block sum.
__device__ __forceinline__ double block_exclusive_scan(double x, double* total)
{
    __shared__ double s_warp[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double inc = x;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const double o = __shfl_up_sync(0xFFFFFFFFu, inc, off);
        if (lane >= off) inc += o;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    double base = 0.0, tot = 0.0;
#pragma unroll
    for (int i = 0; i < SCAN_THREADS / 32; ++i) {
        const double v = s_warp[i];
        if (i < warp) base += v;
        tot += v;
    }
    __syncthreads();
    *total = tot;
    return base + inc - x;
}

__global__ void __launch_bounds__(SCAN_THREADS) psd_terms_kernel(
    const double* __restrict__ psd, double* __restrict__ wfac, double* __restrict__ term,
    double* __restrict__ block_sum, int n_half, int k_lo, double df, double dt, int* err_flag)
{
    const int k0 = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_PER_THREAD;
    double local = 0.0;
#pragma unroll
    for (int i = 0; i < SCAN_PER_THREAD; ++i) {
        const int k = k0 + i;
        if (k >= n_half) break;
        double wf = 0.0, tm = 0.0;
        if (k >= k_lo) {
            const double s = psd[k];
            if (!(s > 0.0)) {
                *err_flag = 1;                       // <= 0 or NaN
            } else if (!isinf(s)) {
                const double f = (double)k * df;
                const double a = pow(f, -7.0 / 6.0);
                wf = 4.0 * df * dt * a / s;
                tm = 4.0 * df * a * a / s;
            }
        }
        wfac[k] = wf;
        term[k] = tm;
        local += tm;
    }
    double total;
    block_exclusive_scan(local, &total);
    if (threadIdx.x == 0) block_sum[blockIdx.x] = total;
}

// In-place exclusive scan of the block totals (at most 2^23 / SCAN_TILE = 8192) by one block.
__global__ void __launch_bounds__(SCAN_THREADS) scan_block_sums_kernel(double* __restrict__ block_sum, int n_blocks)
{
    const int chunk = (n_blocks + SCAN_THREADS - 1) / SCAN_THREADS;
    const int lo = threadIdx.x * chunk, hi = min(n_blocks, lo + chunk);
    double s = 0.0;
    for (int i = lo; i < hi; ++i) s += block_sum[i];
    double total;
    double run = block_exclusive_scan(s, &total);
    for (int i = lo; i < hi; ++i) { const double v = block_sum[i]; block_sum[i] = run; run += v; }
}

__global__ void __launch_bounds__(SCAN_THREADS) prefix_tile_kernel(
    const double* __restrict__ term, const double* __restrict__ block_off, double* __restrict__ prefix, int n_half)
{
    const int k0 = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_PER_THREAD;
    double v[SCAN_PER_THREAD];
    double local = 0.0;
#pragma unroll
    for (int i = 0; i < SCAN_PER_THREAD; ++i) {
        v[i] = (k0 + i < n_half) ? term[k0 + i] : 0.0;
        local += v[i];
    }
    double total;
    double run = block_off[blockIdx.x] + block_exclusive_scan(local, &total);
#pragma unroll
    for (int i = 0; i < SCAN_PER_THREAD; ++i) {
        run += v[i];
        if (k0 + i < n_half) prefix[k0 + i] = run;
    }
}

// ------------------------------------------------------------------ S2: template constants (fp64)
struct SetupArgs {
    const double* __restrict__ bank;     // [n][2] (m1, m2)
    const double* __restrict__ prefix;   // [N/2]
    TemplCoef* __restrict__ coef;        // [n]
    int n_templates;
    int n_half;                          // N/2
    int k_lo;
    double n_over_fs;                    // N / fs  (= 1/df)
    double df;
    float threshold;
    int pn_half_order;                   // 4: 2PN phase (default), 5: + the 2.5PN term
    int* err_flag;
    long long* bad_idx;                  // smallest index of an invalid template (atomicMin), may be null
    unsigned int* tcount;                // [n] per-template trigger counters, zeroed here (may be null)
};

__global__ void template_setup_kernel(const SetupArgs a)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n_templates) return;
    const double m1 = a.bank[2 * i], m2 = a.bank[2 * i + 1];
    if (a.tcount) a.tcount[i] = 0u;
    TemplCoef c;
    c.A1 = c.A2 = c.A3 = c.A5 = 0.0;
    c.k_lo = a.k_lo; c.k_hi = -1;
    c.sigma = c.inv_sigma = 0.f; c.thr2 = 0.f; c.A0 = -0.125f; c.AL = 0.0;
    if (!(m1 > 0.0) || !(m2 > 0.0) || isinf(m1) || isinf(m2)) {
        *a.err_flag = 1;
        if (a.bad_idx) atomicMin(a.bad_idx, (long long)i);
        a.coef[i] = c;
        return;
    }
    const double PI = 3.14159265358979323846;
    const double TSUN = 4.925490947641267e-6;           // G Msun / c^3 [s]
    const double mt = m1 + m2;
    const double M = mt * TSUN;
    const double eta = m1 * m2 / (mt * mt);
    const double f_isco = 1.0 / (pow(6.0, 1.5) * PI * M);
    double khi = floor(f_isco * a.n_over_fs);
    if (khi > (double)(a.n_half - 1)) khi = (double)(a.n_half - 1);
    c.k_hi = (int)khi;
    // Psi_T = -pi/4 + x (b4 + x (b3 + x (b2 + x^2 b0))),  x = f^{-1/3} = df^{-1/3} k^{-1/3}
    const double c0 = 3.0 / (128.0 * eta), p = PI * M;
    const double p13 = cbrt(p);
    const double b0 = c0 / (p * p13 * p13);
    const double b2 = c0 * (3715.0 / 756.0 + 55.0 * eta / 9.0) / p;
    const double b3 = -16.0 * PI * c0 / (p13 * p13);
    const double b4 = c0 * (15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta * eta / 72.0) / p13;
    const double s = 1.0 / cbrt(a.df);
    const double i2pi = 1.0 / (2.0 * PI);
    c.A1 = b4 * s * i2pi;
    c.A2 = b3 * s * s * i2pi;
    c.A3 = b2 * s * s * s * i2pi;
    c.A5 = b0 * s * s * s * s * s * i2pi;
    if (a.pn_half_order >= 5) {
        // NEXT-3 ("order 2.5 in phase"): Psi += c0 pi (38645/756 - 65 eta/9) (1 + 3 ln(v / v_lso)),
        // v_lso = 6^{-1/2} (Arun et al., PRD 71, 084008 (2005), eq. 3.4; Buonanno et al., PRD 80, 084043 (2009),
        // eq. 3.18).  3 ln(v / v_lso) = ln(f / f_ISCO) = ln k + ln(df / f_ISCO): a ln k term and a constant.
        const double B5 = c0 * PI * (38645.0 / 756.0 - 65.0 * eta / 9.0) * i2pi;
        c.AL = B5;
        const double a0 = -0.125 + B5 * (1.0 + log(a.df / f_isco));
        c.A0 = (float)(a0 - rint(a0));
    }
    if (c.k_hi >= c.k_lo) {
        // the generator reduces the phase modulo one cycle with a 2^-32 fixed-point trick that needs
        // |Psi| / 2 pi < 2^19 cycles on the band; |Psi| is largest at k_lo (total masses far below 0.3 Msun at 10 Hz)
        const double ul = 1.0 / cbrt((double)c.k_lo);
        const double ph_lo = fabs(ul * (c.A1 + ul * (c.A2 + ul * (c.A3 + ul * ul * c.A5)))) + fabs(c.AL) * log((double)a.n_half) + 1.0;
        if (!(ph_lo < 524288.0)) {
            *a.err_flag = 1;
            if (a.bad_idx) atomicMin(a.bad_idx, (long long)i);
            c.k_hi = -1;
            a.coef[i] = c;
            return;
        }
        const double sig = sqrt(a.prefix[c.k_hi]);
        c.sigma = (float)sig;
        c.inv_sigma = (float)(1.0 / sig);
        const double th = (double)a.threshold * sig;
        c.thr2 = (float)(th * th);
    }
    a.coef[i] = c;
}

// ------------------------------------------------------------------ triggers: bitonic sort
// Sort by (template, sample).  Tiles of up to TRIG_TILE records are sorted / merged in shared
// memory (trig_sort_tile_kernel); only compare distances >= TRIG_TILE go through global memory
// (trig_bitonic_kernel).  Entries at index >= n are padding (maximal key).
constexpr int TRIG_TILE = 8192;                 // 128 KB of shared memory
__device__ __forceinline__ unsigned long long trig_key(const TrigOut& t)
{
    return ((unsigned long long)(unsigned)t.template_idx << 32) | (unsigned)t.sample_idx;
}
__global__ void trig_bitonic_kernel(TrigOut* trig, long long n_pow2, long long kk, long long jj)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pow2) return;
    const long long ixj = i ^ jj;
    if (ixj > i) {
        const TrigOut a = trig[i], b = trig[ixj];
        const bool up = ((i & kk) == 0);
        const bool gt = trig_key(a) > trig_key(b);
        if (gt == up) { trig[i] = b; trig[ixj] = a; }
    }
}

// tile = min(n_pow2, TRIG_TILE) records per block.  kk_merge == 0: load with padding and run the
// whole network kk = 2..tile; otherwise finish stage kk_merge (jj = tile/2 .. 1).
__global__ void __launch_bounds__(1024) trig_sort_tile_kernel(TrigOut* trig, long long n, int tile, long long kk_merge)
{
    extern __shared__ __align__(16) unsigned char trig_smem_raw[];
    TrigOut* s = reinterpret_cast<TrigOut*>(trig_smem_raw);
    const long long base = (long long)blockIdx.x * tile;
    for (int i = threadIdx.x; i < tile; i += blockDim.x) {
        TrigOut o;
        if (kk_merge != 0 || base + i < n) o = trig[base + i];
        else { o.template_idx = 0x7FFFFFFF; o.sample_idx = 0x7FFFFFFF; o.snr = 0.f; o.phase = 0.f; }
        s[i] = o;
    }
    __syncthreads();
    const long long kk_first = kk_merge ? kk_merge : 2, kk_last = kk_merge ? kk_merge : tile;
    for (long long kk = kk_first; kk <= kk_last; kk <<= 1)
        for (int jj = (int)((kk >> 1) < tile ? (kk >> 1) : (tile >> 1)); jj > 0; jj >>= 1) {
            for (int i = threadIdx.x; i < tile; i += blockDim.x) {
                const int ixj = i ^ jj;
                if (ixj > i) {
                    const TrigOut a = s[i], b = s[ixj];
                    const bool up = (((base + i) & kk) == 0);
                    if ((trig_key(a) > trig_key(b)) == up) { s[i] = b; s[ixj] = a; }
                }
            }
            __syncthreads();
        }
    for (int i = threadIdx.x; i < tile; i += blockDim.x) trig[base + i] = s[i];
}

// Up to TRIG_SMALL records by ONE block: the bitonic network runs on (64-bit key, 16-bit position)
// pairs -- 12 bytes per compare-exchange operand instead of 32 -- with one thread per compare-exchange
// (no idle half), and the 16-byte records are permuted once at the end through shared memory.
constexpr int TRIG_SMALL = 4096;
__global__ void __launch_bounds__(1024) trig_sort_small_kernel(TrigOut* trig, int n, int n_pow2)
{
    extern __shared__ __align__(16) unsigned char trig_smem_raw[];
    unsigned long long* key = reinterpret_cast<unsigned long long*>(trig_smem_raw);          // [n_pow2]
    TrigOut* rec = reinterpret_cast<TrigOut*>(key + n_pow2);                                  // [n_pow2]
    unsigned short* pos = reinterpret_cast<unsigned short*>(rec + n_pow2);                    // [n_pow2]
    for (int i = threadIdx.x; i < n_pow2; i += blockDim.x) {
        unsigned long long k = ~0ULL;                                  // padding sorts last
        if (i < n) { const TrigOut o = trig[i]; rec[i] = o; k = trig_key(o); }
        key[i] = k;
        pos[i] = (unsigned short)i;
    }
    __syncthreads();
    const int n_pairs = n_pow2 >> 1;
    for (int kk = 2; kk <= n_pow2; kk <<= 1)
        for (int jj = kk >> 1; jj > 0; jj >>= 1) {
            for (int p = threadIdx.x; p < n_pairs; p += blockDim.x) {
                const int i = ((p & ~(jj - 1)) << 1) | (p & (jj - 1)), x = i | jj;
                const unsigned long long a = key[i], b = key[x];
                if ((a > b) == ((i & kk) == 0)) {
                    key[i] = b; key[x] = a;
                    const unsigned short t = pos[i]; pos[i] = pos[x]; pos[x] = t;
                }
            }
            __syncthreads();
        }
    for (int i = threadIdx.x; i < n; i += blockDim.x) trig[i] = rec[pos[i]];
}

// The small sort with the count read on the device (the total of the bank's trigger cursor): lets the host enqueue it
// behind the bank without waiting for the count.  Does nothing when there are more triggers than `limit` (the list
// capacity or TRIG_SMALL): the host then takes the general path.
// Fast path (banks of up to TRIG_GROUP_MAX_T templates, no template with more than TRIG_GROUP_MAX_PER triggers -- the
// usual case: a few above-threshold samples per ringing template): the per-template counts the epilogue keeps give
// every template its range by one scan; the records are scattered to their ranges in shared memory and every record
// finds its place by counting the smaller samples of its own range (the threads of a warp mostly share the range, so
// its records are read as broadcasts).  Otherwise the bitonic network of trig_sort_small_kernel.
constexpr int TRIG_GROUP_MAX_T = 8192, TRIG_GROUP_MAX_PER = 1024;
__host__ __device__ constexpr size_t trig_sort_dev_smem()
{
    const size_t bitonic = (sizeof(unsigned long long) + sizeof(TrigOut) + sizeof(unsigned short)) * TRIG_SMALL;
    const size_t group = sizeof(TrigOut) * TRIG_SMALL + 2 * sizeof(int) * (TRIG_GROUP_MAX_T + 1);
    return bitonic > group ? bitonic : group;
}
__global__ void __launch_bounds__(1024) trig_sort_small_dev_kernel(TrigOut* trig, const unsigned long long* __restrict__ cursor,
                                                                   const long long* __restrict__ bad, int limit,
                                                                   const unsigned int* __restrict__ tcount, int n_templates)
{
    extern __shared__ __align__(16) unsigned char trig_smem_raw[];
    __shared__ int s_part[32];
    __shared__ int s_max;
    if (__ldg(bad) != NO_BAD_TEMPLATE) return;
    const unsigned long long found = __ldg(cursor);
    if (found > (unsigned long long)limit || found < 2ULL) return;
    const int n = (int)found;
    if (n_templates <= TRIG_GROUP_MAX_T) {
        TrigOut* rec = reinterpret_cast<TrigOut*>(trig_smem_raw);                             // [TRIG_SMALL]
        int* off = reinterpret_cast<int*>(rec + TRIG_SMALL);                                  // [n_templates + 1] range starts
        int* fill = off + (TRIG_GROUP_MAX_T + 1);                                             // [n_templates] running fill
        // per-thread chunk of the counts: local sum and maximum, block scan of the sums, then the starts
        const int per = (n_templates + (int)blockDim.x - 1) / (int)blockDim.x;
        const int t0 = threadIdx.x * per, t1 = min(n_templates, t0 + per);
        int sum = 0, mx = 0;
        for (int t = t0; t < t1; ++t) { const int cnt = (int)tcount[t]; sum += cnt; mx = max(mx, cnt); }
        int inc = sum;
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xFFFFFFFFu, inc, o); if (lane >= o) inc += v; }
        mx = __reduce_max_sync(0xFFFFFFFFu, mx);
        if (threadIdx.x == 0) s_max = 0;
        if (lane == 31) s_part[warp] = inc;
        __syncthreads();
        if (lane == 0) atomicMax(&s_max, mx);
        if (warp == 0) {
            int v = s_part[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int w = __shfl_up_sync(0xFFFFFFFFu, v, o); if (lane >= o) v += w; }
            s_part[lane] = v;
        }
        __syncthreads();
        if (s_max <= TRIG_GROUP_MAX_PER) {
            int run = inc - sum + (warp > 0 ? s_part[warp - 1] : 0);
            for (int t = t0; t < t1; ++t) { off[t] = run; fill[t] = 0; run += (int)tcount[t]; }
            if (threadIdx.x == 0) off[n_templates] = n;
            __syncthreads();
            for (int i = threadIdx.x; i < n; i += blockDim.x) {
                const TrigOut o = trig[i];
                rec[off[o.template_idx] + atomicAdd(&fill[o.template_idx], 1)] = o;
            }
            __syncthreads();
            for (int i = threadIdx.x; i < n; i += blockDim.x) {                               // rank inside the template's range
                const TrigOut o = rec[i];
                const int a0 = off[o.template_idx], a1 = off[o.template_idx + 1];
                int r = 0;
                for (int j = a0; j < a1; ++j) r += (rec[j].sample_idx < o.sample_idx) ? 1 : 0;
                trig[a0 + r] = o;
            }
            return;
        }
        __syncthreads();
    }
    int n_pow2 = 2;
    while (n_pow2 < n) n_pow2 <<= 1;
    unsigned long long* key = reinterpret_cast<unsigned long long*>(trig_smem_raw);          // [n_pow2]
    TrigOut* rec = reinterpret_cast<TrigOut*>(key + n_pow2);                                  // [n_pow2]
    unsigned short* pos = reinterpret_cast<unsigned short*>(rec + n_pow2);                    // [n_pow2]
    for (int i = threadIdx.x; i < n_pow2; i += blockDim.x) {
        unsigned long long k = ~0ULL;
        if (i < n) { const TrigOut o = trig[i]; rec[i] = o; k = trig_key(o); }
        key[i] = k;
        pos[i] = (unsigned short)i;
    }
    __syncthreads();
    const int n_pairs = n_pow2 >> 1;
    for (int kk = 2; kk <= n_pow2; kk <<= 1)
        for (int jj = kk >> 1; jj > 0; jj >>= 1) {
            for (int p = threadIdx.x; p < n_pairs; p += blockDim.x) {
                const int i = ((p & ~(jj - 1)) << 1) | (p & (jj - 1)), x = i | jj;
                const unsigned long long a = key[i], b = key[x];
                if ((a > b) == ((i & kk) == 0)) {
                    key[i] = b; key[x] = a;
                    const unsigned short t = pos[i]; pos[i] = pos[x]; pos[x] = t;
                }
            }
            __syncthreads();
        }
    for (int i = threadIdx.x; i < n; i += blockDim.x) trig[i] = rec[pos[i]];
}

// ------------------------------------------------------------------ NEXT-4: chi-squared veto (ref. [24])
// Allen's time-frequency discriminator at ONE output sample j per template.  The band [k_lo, k_hi] is cut into p
// contiguous sub-bands of equal expected SNR^2 on the prefix table P (S0): bin k belongs to band
// floor(p P[k-1] / sigma^2), i.e. band l starts at the first bin with P[k-1] >= l sigma^2 / p (reading A26).
//   z_l = sum_{k in band l} w[k] e^{+i Psi(f_k)} e^{+2 pi i jk/N},  sigma_l^2 = P[last bin of l] - P[first bin - 1],
//   chi^2 = sum_l |z_l - p_l z|^2 / (p_l sigma^2),  p_l = sigma_l^2 / sigma^2,  z = sum_l z_l.
// A single sample needs no FFT: the sums are taken directly, one block per (band, template), in double.
constexpr int CHISQ_MAX_BANDS = 256;

__global__ void chisq_edges_kernel(const TemplCoef* __restrict__ coef, const double* __restrict__ prefix, int p,
                                   int* __restrict__ edges /* [n][p + 1] */, int n_templates)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_templates * (p + 1)) return;
    const int b = i / (p + 1), l = i % (p + 1);
    const TemplCoef* tc = coef + b;
    const int k_lo = tc->k_lo, k_hi = tc->k_hi;
    int e = k_hi + 1;
    if (k_hi >= k_lo && l < p) {
        const double sigma2 = prefix[k_hi];
        // smallest k in [k_lo, k_hi] with floor(p P[k-1] / sigma2) >= l  (P[k_lo - 1] = 0); monotone in k
        int lo = k_lo, hi = k_hi + 1;
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            const double run = (mid > k_lo) ? prefix[mid - 1] : 0.0;
            int band = (int)floor(run / sigma2 * (double)p);
            if (band > p - 1) band = p - 1;
            if (band >= l) hi = mid; else lo = mid + 1;
        }
        e = lo;
    }
    edges[i] = e;
}

__global__ void __launch_bounds__(256) chisq_bands_kernel(const c2* __restrict__ w, const double* __restrict__ u,
                                                          const double* __restrict__ lnk,
                                                          const TemplCoef* __restrict__ coef,
                                                          const int* __restrict__ edges, const int* __restrict__ sample_idx,
                                                          int p, int log2n, double* __restrict__ zl /* [n][p][2] */)
{
    const int l = blockIdx.x, b = blockIdx.y;
    const TemplCoef* tc = coef + b;
    const int k0 = edges[b * (p + 1) + l], k1 = edges[b * (p + 1) + l + 1];
    const long long j = sample_idx[b];
    const SpaCoef sc = spa_coef(tc);
    const unsigned long long mask = (1ULL << log2n) - 1ULL;
    const float two_over_n = 2.0f / (float)(1ULL << log2n);
    double sr = 0.0, si = 0.0;
    if (j >= 0) {
        for (int k = k0 + threadIdx.x; k < k1; k += blockDim.x) {
            const c2 q = cmul(__ldg(w + k), spa_phasor_u(__ldg(u + k), k, sc, lnk));
            const c2 r = cmul(q, expi_frac((int)(((unsigned long long)j * (unsigned long long)k) & mask), two_over_n));
            sr += (double)re(r);
            si += (double)im(r);
        }
    }
    __shared__ double s_r[8], s_i[8];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        sr += __shfl_down_sync(0xFFFFFFFFu, sr, off);
        si += __shfl_down_sync(0xFFFFFFFFu, si, off);
    }
    if ((threadIdx.x & 31) == 0) { s_r[threadIdx.x >> 5] = sr; s_i[threadIdx.x >> 5] = si; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tr = 0.0, ti = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) { tr += s_r[i]; ti += s_i[i]; }
        zl[((size_t)b * p + l) * 2] = tr;
        zl[((size_t)b * p + l) * 2 + 1] = ti;
    }
}

__global__ void chisq_finish_kernel(const TemplCoef* __restrict__ coef, const double* __restrict__ prefix,
                                    const int* __restrict__ edges, const double* __restrict__ zl, int p,
                                    float* __restrict__ chisq, int n_templates)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_templates) return;
    const TemplCoef* tc = coef + b;
    float out = 0.f;
    if (tc->k_hi >= tc->k_lo) {
        const double sigma2 = prefix[tc->k_hi];
        double zr = 0.0, zi = 0.0;
        for (int l = 0; l < p; ++l) { zr += zl[((size_t)b * p + l) * 2]; zi += zl[((size_t)b * p + l) * 2 + 1]; }
        double chi = 0.0;
        for (int l = 0; l < p; ++l) {
            const int e0 = edges[b * (p + 1) + l], e1 = edges[b * (p + 1) + l + 1];
            if (e1 <= e0) continue;
            const double s2 = prefix[e1 - 1] - ((e0 > tc->k_lo) ? prefix[e0 - 1] : 0.0);
            const double pl = s2 / sigma2;
            if (!(pl > 0.0)) continue;
            const double er = zl[((size_t)b * p + l) * 2] - pl * zr, ei = zl[((size_t)b * p + l) * 2 + 1] - pl * zi;
            chi += (er * er + ei * ei) / (pl * sigma2);
        }
        out = (float)chi;
    }
    chisq[b] = out;
}

// ------------------------------------------------------------------ diagnostics
__global__ void snr_from_z_kernel(const float2* __restrict__ z, float* __restrict__ snr, size_t n, float inv_sigma)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) snr[i] = sqrtf(fmaf(z[i].x, z[i].x, z[i].y * z[i].y)) * inv_sigma;
}

// h~[k] = f_k^{-7/6} conj(q[k]) for k < N/2 (q = the product generator's e^{+i Psi_T} on the band, zero elsewhere,
// dumped by p1_kernel<LOAD_GEN_DUMP> with unit weights); h~[N/2] = 0.
__global__ void debug_template_kernel(const c2* __restrict__ q, float2* __restrict__ h, int n_half, double df)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > n_half) return;
    float2 o = make_float2(0.f, 0.f);
    if (k >= 1 && k < n_half) {
        const c2 e = q[k];
        const float amp = (float)pow((double)k * df, -7.0 / 6.0);
        o = make_float2(amp * re(e), -amp * im(e));
    }
    h[k] = o;
}

__global__ void fill_ones_kernel(c2* __restrict__ w, int n)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) w[k] = pk(1.0f, 0.0f);
}

// generator alone: q~[b][k] = w[k] e^{+i Psi_b(f_k)}, k < N/2  (config-4 generator throughput)
__global__ void __launch_bounds__(256) generate_only_kernel(const c2* __restrict__ w, const double* __restrict__ u,
                                                            const double* __restrict__ lnk,
                                                            const TemplCoef* __restrict__ coef,
                                                            c2* __restrict__ q, int n_half)
{
    const int b = blockIdx.y;
    const TemplCoef* tc = coef + b;
    const SpaCoef sc = spa_coef(tc);
    const int k_lo = tc->k_lo, k_hi = tc->k_hi;
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n_half; k += gridDim.x * blockDim.x) {
        c2 o = czero();
        if (k >= k_lo && k <= k_hi) o = cmul(__ldg(w + k), spa_phasor_u(__ldg(u + k), k, sc, lnk));
        q[(size_t)b * n_half + k] = o;
    }
}

}  // namespace cbmf
