// td.cuh -- SURVEY.md §8(f) NEXT-3, second part: the paper's OWN template path on sm_100a.
//
//   "the two polarization of the template signal are generated, FFT transformed and normalized ... with a complex
//   product and reduction algorithms"; "order 2.5 in phase and 0 in amplitude";
//   then complex_mf, two inverse transforms and the quadrature sum.
//
// Per template, all on the device:
//   td_setup_kernel     constants of the explicit-in-time chirp (reading A28: "TaylorT3", Blanchet, Living
//                       Rev. Relativity 9, 4 (2006), eq. (234)) and its extent, one thread per template, fp64
//   td_generate_kernel  g[j] = h_+[j] - i h_x[j], one thread per sample (phase in fp64, SFU sine / cosine)
//   p1<LOAD_CPLX> + p2<EPI_STORE>      U = sum_j g[j] e^{+2 pi i jk/N}: both forward transforms in ONE complex FFT,
//                       G[k] = dt conj(U[k]) with g = h_+ + i h_x, H_+ = (G[k] + conj G[N-k]) / 2, H_x = (G[k] - conj G[N-k]) / 2i
//   td_norm_kernel      sigma_p^2 = 4 df sum_k |H_p[k]|^2 / S_n[k]  (block reduction + fp64 atomics)
//   td_product_kernel   P[k], P[N-k]: the two-sided spectrum whose inverse transform is c_+/sigma_+ + i c_x/sigma_x
//   p1<LOAD_CPLX> + p2<EPI_MAX>        rho^2 = |z'|^2, peak and triggers by the epilogue of the SPA path
// The FFT kernels are those of kernels.cuh.  No code is shared with oracle/.
#pragma once
#include "kernels.cuh"

namespace cbmf {

struct __align__(16) TdCoef {
    double theta_per_s;        // eta / (5 M): Theta = tau * theta_per_s
    double cyc;                // (2 / eta) / (2 pi): phi_gw in cycles = -cyc * (x^5 + a2 x^3 - (3 pi/4) x^2 + a4 x + a5 ln Theta), x = Theta^{1/8}
    double a2, a4, a5;
    double tau_start, tau_end; // the template lives on tau_end <= tau <= tau_start (both 0: empty)
    float f_scale_over_flow;   // 1 / (5 pi M f_low): F / f_low = Phi(y) * this
    float pad;
};
static_assert(sizeof(TdCoef) == 64, "TdCoef layout");

// Phi(y) = (5/8) y^3 + (3/8) a2 y^5 - (3 pi/16) y^6 + (1/8) a4 y^7 + a5 y^8 : 5 pi M F, y = Theta^{-1/8}
__device__ __forceinline__ double td_Phi(const double a2, const double a4, const double a5, const double y)
{
    const double y2 = y * y;
    return y2 * y * (0.625 + y2 * (0.375 * a2 + y * (-0.58904862254808623221 + y * (0.125 * a4 + y * a5))));
}
__device__ __forceinline__ double td_dPhi_y2(const double a2, const double a4, const double a5, const double y)   // (dPhi/dy) / y^2
{
    const double y2 = y * y;
    return 1.875 + y2 * (1.875 * a2 + y * (-3.53429173528851739327 + y * (0.875 * a4 + y * 8.0 * a5)));
}
__device__ __forceinline__ double td_root_Phi(const double a2, const double a4, const double a5, double lo, double hi, const double target)
{
    for (int i = 0; i < 200; ++i) {
        const double mid = 0.5 * (lo + hi);
        if (td_Phi(a2, a4, a5, mid) < target) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

struct TdSetupArgs {
    const double* __restrict__ bank;     // [n][2]
    TdCoef* __restrict__ td;             // [n]
    TemplCoef* __restrict__ coef;        // [n] constants of the arg-max epilogue (sigma filled in by td_norm_finish_kernel)
    double* __restrict__ norm;           // [n][2] sigma_+^2, sigma_x^2 accumulators, zeroed here
    unsigned int* tcount;                // [n] trigger counters, zeroed here
    int n_templates, n_half, k_lo, pn_half_order;
    double f_low, seg_seconds;           // N dt
    float threshold;
    int* err_flag;
    long long* bad_idx;
};

__global__ void td_setup_kernel(const TdSetupArgs a)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n_templates) return;
    const double m1 = a.bank[2 * i], m2 = a.bank[2 * i + 1];
    a.norm[2 * i] = a.norm[2 * i + 1] = 0.0;
    if (a.tcount) a.tcount[i] = 0u;
    TdCoef q;
    q.theta_per_s = q.cyc = q.a2 = q.a4 = q.a5 = q.tau_start = q.tau_end = 0.0;
    q.f_scale_over_flow = 0.f; q.pad = 0.f;
    TemplCoef c;
    c.A1 = c.A2 = c.A3 = c.A5 = c.AL = 0.0;
    c.k_lo = a.k_lo; c.k_hi = -1;
    c.sigma = 0.f; c.inv_sigma = 0.f; c.A0 = 0.f;
    const float th = a.threshold;
    c.thr2 = th * th;                                   // rho^2 = |z'|^2 is already normalised
    auto bad = [&]() {
        *a.err_flag = 1;
        if (a.bad_idx) atomicMin(a.bad_idx, (long long)i);
        a.td[i] = q; a.coef[i] = c;
    };
    if (!(m1 > 0.0) || !(m2 > 0.0) || isinf(m1) || isinf(m2)) { bad(); return; }
    const double PI = 3.14159265358979323846, TSUN = 4.925490947641267e-6;
    const double mt = m1 + m2, M = mt * TSUN, eta = m1 * m2 / (mt * mt);
    const double a2 = 3715.0 / 8064.0 + 55.0 * eta / 96.0;
    const double a4 = 9275495.0 / 14450688.0 + 284875.0 * eta / 258048.0 + 1855.0 * eta * eta / 2048.0;
    const double a5 = a.pn_half_order >= 5 ? (-38645.0 / 172032.0 + 65.0 * eta / 2048.0) * PI : 0.0;
    const double scale = 5.0 * PI * M;                  // Phi = scale F
    // y_t: where the frequency stops sweeping upward (smallest positive root of dPhi/dy; 4 if none below it)
    double y_t = 4.0;
    for (int s = 1; s <= 1024; ++s) {
        const double y = (double)s / 256.0;
        if (td_dPhi_y2(a2, a4, a5, y) <= 0.0) {
            double lo = (double)(s - 1) / 256.0, hi = y;
            for (int it = 0; it < 200; ++it) {
                const double mid = 0.5 * (lo + hi);
                if (td_dPhi_y2(a2, a4, a5, mid) > 0.0) lo = mid; else hi = mid;
            }
            y_t = 0.5 * (lo + hi);
            break;
        }
    }
    const double f_isco = 1.0 / (pow(6.0, 1.5) * PI * M);
    const double y_end = (td_Phi(a2, a4, a5, y_t) >= scale * f_isco) ? td_root_Phi(a2, a4, a5, 0.0, y_t, scale * f_isco) : y_t;
    q.theta_per_s = eta / (5.0 * M);
    q.cyc = (2.0 / eta) / (2.0 * PI);
    q.a2 = a2; q.a4 = a4; q.a5 = a5;
    q.f_scale_over_flow = (float)(1.0 / (scale * a.f_low));
    if (td_Phi(a2, a4, a5, y_end) > scale * a.f_low) {
        const double y_start = td_root_Phi(a2, a4, a5, 0.0, y_end, scale * a.f_low);
        const double ys2 = y_start * y_start, ys4 = ys2 * ys2, ye2 = y_end * y_end, ye4 = ye2 * ye2;
        q.tau_start = (5.0 * M / eta) / (ys4 * ys4);
        q.tau_end = (5.0 * M / eta) / (ye4 * ye4);
        // the template must fit the segment, and its phase the 2^19 cycles of the fixed-point reduction
        const double x = 1.0 / y_start, x2 = x * x;
        const double cyc_max = q.cyc * (x2 * x2 * x + a2 * x2 * x + a4 * x + fabs(a5) * 8.0 * fabs(log(y_start))) + 8.0;
        if (!(q.tau_start < a.seg_seconds) || !(cyc_max < 524288.0)) { q.tau_start = q.tau_end = 0.0; bad(); return; }
        c.k_hi = a.n_half - 1;
        c.inv_sigma = 1.f;
    }
    a.td[i] = q;
    a.coef[i] = c;
}

// g[b][j] = (F/f_low)^{2/3} (cos phi_gw, sign * sin phi_gw) at tau_j = (N - j) dt (j = 0: N dt); zero outside the
// template's extent.  sign = -1: the conjugate, input of the forward transform; +1: the polarisations themselves.
__global__ void __launch_bounds__(256) td_generate_kernel(const TdCoef* __restrict__ td, c2* __restrict__ g, int n, double dt, float sign)
{
    const int b = blockIdx.y;
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const TdCoef q = td[b];
    const double tau = (double)(n - j) * dt;
    c2 o = czero();
    if (q.tau_start > 0.0 && tau <= q.tau_start && tau >= q.tau_end) {
        const double theta = tau * q.theta_per_s;
        const double x = sqrt(sqrt(sqrt(theta)));                    // Theta^{1/8} = 1 / y
        const double x2 = x * x;
        double s = fma(x2, x2 * x, q.a2 * (x2 * x));
        s = fma(-2.35619449019234492885, x2, s);
        s = fma(q.a4, x, s);
        if (q.a5 != 0.0) s = fma(q.a5, log(theta), s);
        const double ph = -q.cyc * s;                                // cycles, |ph| < 2^19 (td_setup_kernel)
        const int frac = __double2loint(__dadd_rn(ph, 1572864.0));
        const float ang = (float)frac * (6.28318530717958647692f / 4294967296.0f);
        const float y = (float)(1.0 / x);
        const float y2 = y * y;
        const float phi = y2 * y * (0.625f + y2 * (0.375f * (float)q.a2 + y * (-0.58904862254808623221f + y * (0.125f * (float)q.a4 + y * (float)q.a5))));
        const float amp = exp2f(0.66666666666666667f * log2f(phi * q.f_scale_over_flow));
        o = pk(amp * __cosf(ang), sign * amp * __sinf(ang));
    }
    g[(size_t)b * n + j] = o;
}

// winv[k] = 4 df / S_n[k] and wd[k] = 4 df d~[k] / S_n[k] (zero outside [k_lo, N/2) and where S_n = inf), from the
// S0 / S1 tables wfac = 4 df dt f^{-7/6} / S_n and w = 4 df d~ f^{-7/6} / S_n.
__global__ void td_tables_kernel(const double* __restrict__ wfac, const c2* __restrict__ w, float* __restrict__ winv,
                                 c2* __restrict__ wd, int n_half, int k_lo, double df, double dt)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_half) return;
    float wi = 0.f;
    c2 o = czero();
    if (k >= k_lo) {
        const double f76 = pow((double)k * df, 7.0 / 6.0);
        wi = (float)(wfac[k] * f76 / dt);
        const c2 wk = w[k];
        o = pk((float)((double)re(wk) * f76), (float)((double)im(wk) * f76));
    }
    winv[k] = wi;
    wd[k] = o;
}

// sigma_+^2 and sigma_x^2 of template b from U = sum_j conj(g)[j] e^{+2 pi i jk/N}:  with A = dt conj(U[k]) = G[k] and
// B = dt U[N-k] = conj(G[N-k]):  H_+ = (A + B)/2,  H_x = (A - B)/(2i);  sigma_p^2 = sum_k winv[k] |H_p[k]|^2.
__global__ void __launch_bounds__(256) td_norm_kernel(const c2* __restrict__ U, const float* __restrict__ winv,
                                                      double* __restrict__ norm, int n, int k_lo, float dt)
{
    const int b = blockIdx.y;
    const c2* __restrict__ u = U + (size_t)b * n;
    double sp = 0.0, sc = 0.0;
    for (int k = k_lo + blockIdx.x * blockDim.x + threadIdx.x; k < n / 2; k += gridDim.x * blockDim.x) {
        float ux, uy, vx, vy;
        unpk(u[k], ux, uy);
        unpk(u[n - k], vx, vy);
        // A = dt (ux, -uy), B = dt (vx, vy)
        const float px = dt * (ux + vx), py = dt * (vy - uy);        // A + B
        const float mx = dt * (ux - vx), my = dt * (-uy - vy);       // A - B
        const float wi = 0.25f * winv[k];
        sp += (double)(wi * fmaf(px, px, py * py));
        sc += (double)(wi * fmaf(mx, mx, my * my));
    }
    __shared__ double s_p[8], s_c[8];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        sp += __shfl_down_sync(0xFFFFFFFFu, sp, off);
        sc += __shfl_down_sync(0xFFFFFFFFu, sc, off);
    }
    if ((threadIdx.x & 31) == 0) { s_p[threadIdx.x >> 5] = sp; s_c[threadIdx.x >> 5] = sc; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tp = 0.0, tc = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) { tp += s_p[i]; tc += s_c[i]; }
        atomicAdd(norm + 2 * b, tp);
        atomicAdd(norm + 2 * b + 1, tc);
    }
}

// sigma_+ into the epilogue's constants; a template without power in the band becomes an empty one.
__global__ void td_norm_finish_kernel(const double* __restrict__ norm, TemplCoef* __restrict__ coef, float2* __restrict__ inv_sig, int n_templates)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_templates) return;
    const double sp = sqrt(norm[2 * b]), sc = sqrt(norm[2 * b + 1]);
    float2 o = make_float2(0.f, 0.f);
    if (coef[b].k_hi >= coef[b].k_lo && sp > 0.0 && sc > 0.0) {
        o = make_float2((float)(1.0 / sp), (float)(1.0 / sc));
        coef[b].sigma = (float)sp;
    } else {
        coef[b].k_hi = -1; coef[b].sigma = 0.f; coef[b].inv_sigma = 0.f;
    }
    inv_sig[b] = o;
}

// In place U -> P: with X = conj(A) + conj(B) = 2 conj(H_+), V = conj(A) - conj(B) (conj(H_x) = i V / 2), Q_p = wd conj(H_p) / sigma_p:
//   P[k]   = (Q_+ + i Q_x) / 2           = wd       [X / (4 sigma_+) - V / (4 sigma_x)]
//   P[N-k] = (conj Q_+ + i conj Q_x) / 2 = conj(wd) [conj(X) / (4 sigma_+) + conj(V) / (4 sigma_x)]
// so that sum_k P[k] e^{+2 pi i jk/N} = Re(...)_+ + i Re(...)_x = c_+[j]/sigma_+ + i c_x[j]/sigma_x.  Zero outside [k_lo, N/2).
__global__ void __launch_bounds__(256) td_product_kernel(c2* __restrict__ U, const c2* __restrict__ wd, const float2* __restrict__ inv_sig,
                                                         int n, int k_lo, float dt)
{
    const int b = blockIdx.y;
    c2* __restrict__ u = U + (size_t)b * n;
    const float2 is = inv_sig[b];
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k <= n / 2; k += gridDim.x * blockDim.x) {
        if (k < k_lo || k == n / 2 || k == 0) {
            u[k] = czero();
            if (k > 0 && k < n / 2) u[n - k] = czero();
            continue;
        }
        float ux, uy, vx, vy, wx, wy;
        unpk(u[k], ux, uy);
        unpk(u[n - k], vx, vy);
        unpk(wd[k], wx, wy);
        // conj(A) = dt (ux, uy), conj(B) = dt (vx, -vy)
        const float Xx = dt * (ux + vx), Xy = dt * (uy - vy);
        const float Vx = dt * (ux - vx), Vy = dt * (uy + vy);
        const float sp = 0.25f * is.x, sc = 0.25f * is.y;
        const float ax = Xx * sp - Vx * sc, ay = Xy * sp - Vy * sc;          // X/(4 s+) - V/(4 sx)
        const float bx = Xx * sp + Vx * sc, by = -(Xy * sp + Vy * sc);       // conj(X)/(4 s+) + conj(V)/(4 sx)
        u[k] = pk(wx * ax - wy * ay, wx * ay + wy * ax);
        u[n - k] = pk(wx * bx + wy * by, wx * by - wy * bx);                  // conj(wd) * (bx, by)
    }
}

// (h_+, h_x)[j] from the generated g with sign = +1 (diagnostic)
__global__ void td_copy_kernel(const c2* __restrict__ g, float2* __restrict__ h, int n)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) h[j] = make_float2(re(g[j]), im(g[j]));
}

}  // namespace cbmf
