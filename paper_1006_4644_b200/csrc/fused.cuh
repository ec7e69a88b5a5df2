// fused.cuh -- the whole bank in ONE persistent launch.
//
// bank_kernel<L1, L2> runs one block of 512 threads per SM (cooperative launch: every block is
// resident) and walks the bank with two kinds of work, scheduled inside the kernel:
//
//   P1 (tile, template)   SPA generation + correlate + N1-point column FFTs of NC adjacent
//                         columns k2 -> Y[slot][j1][k2].  Tile `i` belongs to block `i`, which
//                         stages w[k] and k^{-1/3} of its columns in shared memory ONCE per
//                         launch and then takes the templates in order, two at a time (one per
//                         half of the block, each half with its own exchange buffer and named
//                         barrier).
//   P2 (template, rows)   twiddle + N2-point row FFTs + |z|^2 + arg-max / threshold of 64
//                         adjacent rows j1 (16 warps x 4 rows), claimed from a global queue by
//                         any block, as soon as all tiles of that template have been written.
//
// Y is a ring of `ring` templates (8 N bytes each) so that the inter-pass buffer stays in the
// L2 cache: P1 may write template b only when P2 has finished template b - ring.
//
// Progress: a block never waits while holding work -- it takes a P1 step only when the ring slot
// is free and claims a P2 item only when its template is complete -- so the earliest unfinished
// template can always advance.  Every wait is bounded; on a timeout the abort flag stops all blocks
// and the host reports CBMF_ECUDA instead of hanging.
//
// Ordering (release / acquire at gpu scope): a half block finishes its stores of Y, meets at its
// barrier, and one thread fences and increments p1_done[b]; the claiming thread reads the counter
// with ld.acquire and the block barrier hands the ordering to the other threads, which read Y
// with cp.async.cg (L2, never a stale L1 line).  The same pattern in the other direction frees a
// ring slot (p2_done[b]).
#pragma once
#include "kernels.cuh"

namespace cbmf {

struct FusedArgs {
    const c2* __restrict__ w;              // [N/2]
    const double* __restrict__ u;          // [N/2]
    const TemplCoef* __restrict__ coef;    // [n_templates]
    c2* Y;                                 // [ring][N]
    c2* cand;                              // [ring][N / E2]
    unsigned long long* best_key;          // [n_templates], zero on entry
    unsigned int* p1_done;                 // [n_templates], zero on entry: tiles written
    unsigned int* done_ctr;                // [n_templates], zero on entry: P2 items past the epilogue
    unsigned int* p2_done;                 // [n_templates], zero on entry: P2 items that released the slot
    unsigned int* p2_next;                 // [1], zero on entry: next P2 item of the queue
    int* abort_flag;                       // [1], zero on entry
    PeakOut* peaks;                        // [n_templates]
    TrigOut* trig;
    unsigned long long* trig_cursor;
    unsigned long long trig_cap;
    int n_templates;
    int ring;                              // even, >= 2
    unsigned long long* stats;             // null, or [grid][6]: cycles deciding / in P1 / in P2, steps P1 / P2, total
    int p2_first;                          // scheduling: 1 = a ready P2 item is preferred to the next P1 step
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ int ld_volatile_s32(const int* p)
{
    int v;
    asm volatile("ld.volatile.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

template <int L1, int L2>
struct FusedCfg {
    using C1 = Cfg<L1>;
    using C2 = Cfg<L2>;
    static constexpr int NT = 512;
    static constexpr int HALF = 256;                                   // threads of one P1 half
    static constexpr int NC = HALF / C1::T;                            // columns per tile
    static constexpr int NTILES = L2 / NC;
    static constexpr int ROWS = NT / C2::T;                            // rows in flight in P2
    static constexpr int RPW = 4;                                      // rows per row group and item
    static constexpr int ITEM_ROWS = ROWS * RPW;
    static constexpr int ITEMS2 = L1 / ITEM_ROWS;                      // P2 items per template
    static constexpr size_t EX_HALF = (size_t)C1::PADDED * NC;         // c2 per P1 exchange buffer
    static constexpr size_t P2_ELEMS = (size_t)p2_row_stride<L2>() * ROWS;
    static constexpr size_t REGION_A = (2 * EX_HALF > P2_ELEMS) ? 2 * EX_HALF : P2_ELEMS;
    static constexpr size_t W_ELEMS = (size_t)(L1 / 2) * NC;           // c2 (w tile) and double (u tile)
    static constexpr size_t TW_ELEMS = (size_t)twtab_elems<L1>();
    static constexpr size_t SMEM_BYTES = sizeof(c2) * (REGION_A + W_ELEMS + TW_ELEMS) + sizeof(double) * W_ELEMS;
    static_assert(C1::R3 == 1, "fused kernel: two-step column FFT");
    static_assert(C2::T <= 32, "fused kernel: one warp per row");
    static_assert(C1::T * NC == HALF && L1 % ITEM_ROWS == 0, "fused kernel geometry");
};

// One template of one tile by one half of the block (256 threads, lt = thread index in the half).
template <int L1, int L2>
__device__ __forceinline__ void fused_p1(const FusedArgs& a, const int tile, const int b, const int lt,
                                         const int bar_id, c2* __restrict__ ex, const c2* __restrict__ wt,
                                         const double* __restrict__ ut, const c2* __restrict__ tw,
                                         const TemplCoef* __restrict__ tc)
{
    using F = FusedCfg<L1, L2>;
    using C = Cfg<L1>;
    constexpr int E = C::E, T = C::T, R1 = C::R1, NC = F::NC, RL = C::R2;
    constexpr int NZ1 = R1 / 2;                                        // bins k >= N/2 are zero
    constexpr size_t n_total = (size_t)L1 * L2;
    const int c = lt % NC, t = lt / NC;
    const int k2 = tile * NC + c;

    c2 v[E];
    spa_correlate<L1, L2>(v, t, k2, wt + c, NC, ut + c, NC, tc->k_lo, tc->k_hi, tc->A1, tc->A2, tc->A3, tc->A5);

    fft_core<L1, NZ1, NC, SYNC_NAMED, false>(v, t, ex + c, 0, 1, NoHook(), tw, bar_id, F::HALF);

    c2* __restrict__ yb = a.Y + (size_t)(b % a.ring) * n_total + y_index<L1, NC>(t, k2);
#pragma unroll
    for (int u = 0; u < E / RL; ++u)
#pragma unroll
        for (int q = 0; q < RL; ++q)
            yb[(size_t)(T * u + (L1 / RL) * q) * NC] = v[u * RL + q];      // row j1 = t + T u + (L1/RL) q
    named_barrier(bar_id, F::HALF);      // exchange buffer free again; every store of the half issued
    if (lt == 0) {
        __threadfence();
        atomicAdd(a.p1_done + b, 1u);
    }
}

// One P2 item: rows [rb * ITEM_ROWS, +ITEM_ROWS) of template b, all 512 threads.
template <int L1, int L2>
__device__ __forceinline__ void fused_p2(const FusedArgs& a, const int b, const int rb, c2* __restrict__ smem)
{
    using F = FusedCfg<L1, L2>;
    using C = Cfg<L2>;
    constexpr int T = C::T, ROWS = F::ROWS, RPW = F::RPW;
    constexpr int LG1 = ilog2c(L1);
    constexpr size_t n_total = (size_t)L1 * L2;
    const int slot = b % a.ring;
    P2Args p;
    p.Y = a.Y + (size_t)slot * n_total;
    p.coef = a.coef + b;
    p.best_key = a.best_key + b;
    p.cand = a.cand + (size_t)slot * (n_total / C::E);
    p.done_ctr = nullptr; p.peaks = nullptr;
    p.trig = a.trig; p.trig_cursor = a.trig_cursor; p.trig_cap = a.trig_cap;
    p.tmpl_base = b;
    p.z_out = nullptr; p.w_out = nullptr; p.wfac = nullptr;

    const int t = threadIdx.x % T, row = threadIdx.x / T;
    c2* sm = smem + row * p2_row_stride<L2>();
    const int j1_0 = rb * F::ITEM_ROWS + row;
    p2_prefetch_row<L1, L2>(sm, p.Y, j1_0, t);
#pragma unroll 1
    for (int it = 0; it < RPW; ++it) {
        const int j1 = j1_0 + it * ROWS;
        p2_row<L1, L2, EPI_MAX>(p, j1, 0, t, sm, p.Y, (it + 1 < RPW) ? j1 + ROWS : -1);
    }
    __syncthreads();                                 // every row of the item has published and left Y
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned prev = atomicAdd(a.done_ctr + b, 1u);
        if (prev == (unsigned)F::ITEMS2 - 1u) {      // last item of the template: emit the peak record
            __threadfence();
            const TemplCoef* tc = a.coef + b;
            const unsigned long long bk = __ldcg(a.best_key + b);
            PeakOut o;
            if (tc->k_hi < tc->k_lo) {               // empty band
                o.snr_max = 0.f; o.idx_peak = -1; o.phase = 0.f; o.sigma = 0.f;
            } else {
                const float pmax = __uint_as_float((unsigned)(bk >> 32));
                const int j = (int)(0xFFFFFFFFu - (unsigned)(bk & 0xFFFFFFFFu));
                const int j1 = j & (L1 - 1), tt = (j >> LG1) & (T - 1);
                const c2 z = __ldcg(p.cand + (size_t)j1 * T + tt);
                o.snr_max = sqrtf(pmax) * tc->inv_sigma;
                o.idx_peak = j;
                o.phase = atan2f(im(z), re(z));
                o.sigma = tc->sigma;
            }
            a.peaks[b] = o;
            __threadfence();
        }
        atomicAdd(a.p2_done + b, 1u);                // releases the ring slot once all items are here
    }
}

template <int L1, int L2>
__global__ void __launch_bounds__(512, 1) bank_kernel(const FusedArgs a)
{
    extern __shared__ __align__(16) c2 smem[];
    using F = FusedCfg<L1, L2>;
    using C = Cfg<L1>;
    constexpr int NC = F::NC;
    __shared__ int s_act[3];                         // action, template, row block

    c2* __restrict__ wt = smem + F::REGION_A;                                    // [L1/2][NC]
    c2* __restrict__ tw = wt + F::W_ELEMS;                                       // [R1][R2 + 2]
    double* __restrict__ ut = reinterpret_cast<double*>(tw + F::TW_ELEMS);       // [L1/2][NC]

    const int tid = threadIdx.x;
    const int my_tile = ((int)blockIdx.x < F::NTILES) ? (int)blockIdx.x : -1;
    const int nt = a.n_templates;
    if (my_tile >= 0) {
        // stage this block's columns of w and k^{-1/3}: rows of NC * 8 bytes = NC/2 chunks of 16 bytes
        constexpr int CPR = NC / 2, NCHUNK = (L1 / 2) * CPR;
        for (int ci = tid; ci < NCHUNK; ci += F::NT) {
            const int row = ci / CPR, part = ci % CPR;
            const size_t g = (size_t)row * L2 + my_tile * NC + 2 * part;
            cp_async16(wt + row * NC + 2 * part, a.w + g);
            cp_async16(ut + row * NC + 2 * part, a.u + g);
        }
        cp_async_commit();
        twtab_fill<L1>(tw, tid, F::NT);
        cp_async_wait_all();
    }
    __syncthreads();

    const unsigned total2 = (unsigned)nt * (unsigned)F::ITEMS2;
    int next_b1 = (my_tile >= 0) ? 0 : nt;           // next template pair of this block's tile
    bool q_empty = false;                            // the P2 queue has been seen exhausted

    unsigned long long st_dec = 0, st_p1 = 0, st_p2 = 0, n_p1 = 0, n_p2 = 0;
    const long long t_begin = clock64();
    for (;;) {
        const long long t0 = clock64();
        if (tid == 0) {
            int act = 0, tb = 0, rb = 0;             // 0 = exit, 1 = P1 pair, 2 = P2 item, 3 = abort
            unsigned spins = 0;
            for (;;) {
                // (a) the next P1 step of this block's tile, if its ring slots are free (pairs are ring-aligned)
                bool p1_ok = false;
                if (next_b1 < nt) {
                    p1_ok = true;
                    if (next_b1 >= a.ring) {
                        p1_ok = ld_acquire_u32(a.p2_done + (next_b1 - a.ring)) == (unsigned)F::ITEMS2;
                        if (p1_ok && next_b1 + 1 < nt)
                            p1_ok = ld_acquire_u32(a.p2_done + (next_b1 + 1 - a.ring)) == (unsigned)F::ITEMS2;
                    }
                    if (p1_ok && !a.p2_first) { act = 1; tb = next_b1; break; }
                }
                // (b) the item at the head of the P2 queue, if its template is complete
                if (!q_empty) {
                    const unsigned cur = ld_acquire_u32(a.p2_next);
                    if (cur >= total2) {
                        q_empty = true;
                    } else {
                        const int b = (int)(cur / (unsigned)F::ITEMS2);
                        if (ld_acquire_u32(a.p1_done + b) == (unsigned)F::NTILES) {
                            if (atomicCAS(a.p2_next, cur, cur + 1u) == cur) {
                                act = 2; tb = b; rb = (int)(cur % (unsigned)F::ITEMS2);
                                break;
                            }
                            continue;                // lost the race: look again at once
                        }
                    }
                }
                if (p1_ok) { act = 1; tb = next_b1; break; }
                if (q_empty && next_b1 >= nt) { act = 0; break; }
                if (ld_volatile_s32(a.abort_flag) != 0) { act = 3; break; }
                if (++spins > (1u << 22)) { atomicExch(a.abort_flag, 1); act = 3; break; }
                __nanosleep(200);
            }
            s_act[0] = act; s_act[1] = tb; s_act[2] = rb;
        }
        __syncthreads();
        const int act = s_act[0], tb = s_act[1], rb = s_act[2];      // rewritten only after the barrier that ends the step
        const long long t1 = clock64();
        st_dec += (unsigned long long)(t1 - t0);
        if (act == 0 || act == 3) break;
        if (act == 1) {
            const int half = tid / F::HALF, lt = tid % F::HALF;
            const int b = tb + half;
            if (b < nt)
                fused_p1<L1, L2>(a, my_tile, b, lt, 1 + half, smem + (size_t)half * F::EX_HALF, wt, ut, tw, a.coef + b);
            next_b1 = tb + 2;
            __syncthreads();                         // region A is shared with the P2 role
            st_p1 += (unsigned long long)(clock64() - t1); ++n_p1;
        } else {
            fused_p2<L1, L2>(a, tb, rb, smem);
            __syncthreads();
            st_p2 += (unsigned long long)(clock64() - t1); ++n_p2;
        }
    }
    if (a.stats != nullptr && tid == 0) {
        unsigned long long* o = a.stats + 6 * (size_t)blockIdx.x;
        o[0] = st_dec; o[1] = st_p1; o[2] = st_p2; o[3] = n_p1; o[4] = n_p2;
        o[5] = (unsigned long long)(clock64() - t_begin);
    }
}

}  // namespace cbmf
