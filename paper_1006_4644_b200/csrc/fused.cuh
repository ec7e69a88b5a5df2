// fused.cuh -- the whole bank in ONE persistent launch.
//
// bank_kernel<L1, L2> runs two blocks of 256 threads on every SM (cooperative launch: every block
// is resident for the whole bank) and gives each block ONE role for its lifetime:
//
//   P1 block (one per column tile, the first block to arrive on an SM takes a tile):
//       stages w[k] of its NC columns and the generator / twiddle tables in shared memory ONCE,
//       then for template b = 0, 1, ...: SPA generation + correlate + N1-point column FFTs ->
//       output tile in shared memory -> one TMA bulk store into Y[b mod ring] (the body of
//       p1_kernel), and publishes p1_done[b] once that store has completed.
//   P2 block (every other block): claims (template, 64 rows) items from a global queue in order,
//       waits until all tiles of the template have been written, and runs twiddle + N2-point row
//       FFTs + |z|^2 + arg-max / threshold on them (the body of p2_kernel); the last item of a
//       template emits its peak record; every item then frees its share of the ring slot.
//
// So every SM that owns a tile runs one P1 block (generator: FP64 / SFU / shared memory; butterflies:
// FMA pipe) next to one P2 block (FMA-bound), which is the pairing the launch-pair path only gets
// by chance.  Y is a ring of `ring` templates: P1 may write template b only when P2 has finished
// template b - ring.
//
// Progress: P1 blocks wait only for ring slots (freed by P2 items of earlier templates), P2 blocks
// only for P1 of the template they hold (earlier than anything P1 is waiting for): a bounded
// buffer, no cycle.  Every wait is bounded; on a timeout the abort flag stops all blocks and the
// host reports CBMF_ECUDA instead of hanging.
//
// Ordering (release / acquire at gpu scope): the P1 thread that issued the bulk store waits for
// its completion (cp.async.bulk.wait_group), fences and increments p1_done[b]; the claiming P2
// thread reads the counter with ld.acquire and the block barrier hands the ordering to the other
// threads, which read Y with cp.async.cg (L2, never a stale L1 line).  The same pattern in the
// other direction frees a ring slot (p2_done[b]).
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
    unsigned int* tile_next;               // [1], zero on entry: next column tile without a P1 block
    unsigned int* sm_slot;                 // [n_sm], zero on entry: blocks that have arrived on each SM
    int* abort_flag;                       // [1], zero on entry
    PeakOut* peaks;                        // [n_templates]
    TrigOut* trig;
    unsigned long long* trig_cursor;
    unsigned long long trig_cap;
    int n_templates;
    int ring;                              // >= 2
    int use_series;                        // generator: k^{-1/3} by the series of spa_correlate
    unsigned long long* stats;             // null, or [grid][6]: role (1 / 2), cycles waiting, cycles working, steps, total, tile
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
__device__ __forceinline__ unsigned smid()
{
    unsigned v;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(v));
    return v;
}
// At most `n` of this thread's bulk stores are still in flight (their global writes not yet complete).
template <int N_PENDING>
__device__ __forceinline__ void bulk_store_wait_done()
{
    asm volatile("cp.async.bulk.wait_group %0;\n" ::"n"(N_PENDING) : "memory");
}

// Release increment of a counter without a return value: earlier writes this thread has observed
// (here: the completed bulk stores) are visible to whoever acquires the new value.
__device__ __forceinline__ void red_release_add(unsigned* p, const unsigned v)
{
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

template <int L1, int L2>
struct FusedCfg {
    using C1 = Cfg<L1>;
    using C2 = Cfg<L2>;
    static constexpr int NT = 256;
    static constexpr int NC = C1::C;                                   // columns per tile
    static constexpr int NTILES = L2 / NC;
    static constexpr int ROWS = NT / C2::T;                            // rows in flight in a P2 block
    static constexpr int RPW = p2_rpw<L1, L2>();                       // rows per warp and item
    static constexpr int ITEM_ROWS = ROWS * RPW;
    static constexpr int ITEMS2 = L1 / ITEM_ROWS;                      // P2 items per template
    static constexpr size_t P1_BYTES = p1_smem_bytes<L1, LOAD_GEN>();
    static constexpr size_t P2_BYTES = sizeof(c2) * (size_t)p2_row_stride<L2>() * ROWS;
    static constexpr size_t SMEM_BYTES = P1_BYTES > P2_BYTES ? P1_BYTES : P2_BYTES;
    static_assert(C1::NT1 == NT && C2::NT2 == NT, "fused kernel: 256-thread blocks in both roles");
    static_assert(C2::T <= 32, "fused kernel: one warp per row");
    static_assert(L1 % ITEM_ROWS == 0, "fused kernel geometry");
};

// Bounded wait of one thread until *ctr == want (acquire).  false: timed out or another block aborted.
__device__ __forceinline__ bool wait_counter(const unsigned* ctr, const unsigned want, int* abort_flag)
{
    unsigned spins = 0;
    while (ld_acquire_u32(ctr) != want) {
        if (ld_volatile_s32(abort_flag) != 0) return false;
        if (++spins > (1u << 22)) { atomicExch(abort_flag, 1); return false; }
        __nanosleep(100);
    }
    return true;
}

// ---------------------------------------------------------------------------------------- P1 role
// All templates of the bank for column tile `tile` (the loop body is p1_kernel<LOAD_GEN>'s).
template <int L1, int L2>
__device__ __forceinline__ void fused_p1_role(const FusedArgs& a, const int tile, c2* __restrict__ smem,
                                              unsigned long long& st_wait, unsigned long long& n_steps)
{
    using F = FusedCfg<L1, L2>;
    using C = Cfg<L1>;
    constexpr int E = C::E, T = C::T, R1 = C::R1, NC = C::C, NT = F::NT;
    constexpr int RL = (C::R3 > 1) ? C::R3 : C::R2;
    constexpr int NZ1 = R1 / 2;                                        // bins k >= N/2 are zero
    constexpr size_t n_total = (size_t)L1 * L2;
    constexpr bool TWTAB = p1_use_twtab<L1>();
    __shared__ __align__(16) TemplCoef s_coef[2];
    __shared__ int s_ok;

    const int tid = threadIdx.x, nt = a.n_templates;
    const int c = tid % NC, t = tid / NC;
    const int k2 = tile * NC + c;
    c2* __restrict__ tw = smem + (size_t)C::PADDED * NC;
    c2* __restrict__ wt = tw + (TWTAB ? twtab_elems<L1>() : 0);
    double* __restrict__ ub = reinterpret_cast<double*>(wt + (size_t)(L1 / 2) * NC);
    float* __restrict__ inv = reinterpret_cast<float*>(ub + L1 / 2);
    {
        constexpr int CPR = NC / 2, NCHUNK = (L1 / 2) * CPR;
        for (int ci = tid; ci < NCHUNK; ci += NT) {
            const int row = ci / CPR, part = ci % CPR;
            cp_async16(wt + row * NC + 2 * part, a.w + ((size_t)row * L2 + tile * NC + 2 * part));
        }
        if (tid < 4) cp_async16(reinterpret_cast<char*>(&s_coef[0]) + 16 * tid, reinterpret_cast<const char*>(a.coef) + 16 * tid);
        cp_async_commit();
        if constexpr (TWTAB) twtab_fill<L1>(tw, tid, NT);
        for (int k1 = tid; k1 < L1 / 2; k1 += NT) {
            const int kb = k1 * L2 + tile * NC;
            ub[k1] = __ldg(a.u + kb);
            inv[k1] = kb > 0 ? (float)(1.0 / (double)kb) : 0.f;
        }
        cp_async_wait_all();
    }
    __syncthreads();

    int cur = 0, b = 0;
    for (; b < nt; ++b, cur ^= 1) {
        if (tid < 4 && b + 1 < nt)
            cp_async16(reinterpret_cast<char*>(&s_coef[cur ^ 1]) + 16 * tid,
                       reinterpret_cast<const char*>(a.coef + b + 1) + 16 * tid);
        cp_async_commit();
        const TemplCoef* tc = &s_coef[cur];
        c2 v[E];
        if (a.use_series)
            spa_correlate<L1, L2, true>(v, t, k2, wt + c, NC, nullptr, 0, tc->k_lo, tc->k_hi, tc->A1, tc->A2, tc->A3,
                                        tc->A5, ub, inv, (float)c);
        else
            spa_correlate<L1, L2>(v, t, k2, wt + c, NC, a.u + k2, L2, tc->k_lo, tc->k_hi, tc->A1, tc->A2, tc->A3, tc->A5);

        if (tid == 0) {
            int ok = 1;
            if (b >= a.ring) {                       // ring slot of template b: P2 must be through with b - ring
                const long long t0 = clock64();
                ok = wait_counter(a.p2_done + (b - a.ring), (unsigned)F::ITEMS2, a.abort_flag) ? 1 : 0;
                st_wait += (unsigned long long)(clock64() - t0);
            }
            bulk_store_wait_read();                  // the previous output tile has left the exchange buffer
            s_ok = ok;
        }
        __syncthreads();
        if (!s_ok) break;
        fft_core<L1, NZ1, NC, SYNC_BLOCK, false>(v, t, smem + c, 0, 1, NoHook(), TWTAB ? tw : nullptr);

        __syncthreads();                             // every step-2 read of the exchange buffer is done
        c2* __restrict__ ot = smem + (size_t)t * NC + c;
#pragma unroll
        for (int u = 0; u < E / RL; ++u)
#pragma unroll
            for (int q = 0; q < RL; ++q)
                ot[(size_t)(T * u + (L1 / RL) * q) * NC] = v[u * RL + q];      // row j1 = t + T u + (L1/RL) q
        fence_async_smem();
        cp_async_wait_all();                         // the next template's constants have landed
        __syncthreads();
        if (tid == 0) {
            if (b > 0) {                             // the store of template b - 1, issued a whole step ago: publish it
                bulk_store_wait_done<0>();
                red_release_add(a.p1_done + (b - 1), 1u);
            }
            bulk_store(a.Y + (size_t)(b % a.ring) * n_total + (size_t)tile * L1 * NC, smem, (unsigned)(sizeof(c2) * L1 * NC));
        }
        ++n_steps;
    }
    if (tid == 0) {
        bulk_store_wait_done<0>();
        if (b == nt && nt > 0) red_release_add(a.p1_done + (nt - 1), 1u);
    }
}

// ---------------------------------------------------------------------------------------- P2 role
// One item: rows [rb * ITEM_ROWS, +ITEM_ROWS) of template b, by the 8 warps of the block.
template <int L1, int L2>
__device__ __forceinline__ void fused_p2_item(const FusedArgs& a, const int b, const int rb, c2* __restrict__ smem)
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
    P2Tw<L1, L2> rtw;
    rtw.init(j1_0, ROWS, t);
#pragma unroll 1
    for (int it = 0; it < RPW; ++it) {
        const int j1 = j1_0 + it * ROWS;
        p2_row<L1, L2, EPI_MAX>(p, j1, 0, t, sm, p.Y, (it + 1 < RPW) ? j1 + ROWS : -1, rtw);
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
__device__ __forceinline__ void fused_p2_role(const FusedArgs& a, c2* __restrict__ smem,
                                              unsigned long long& st_wait, unsigned long long& n_steps)
{
    using F = FusedCfg<L1, L2>;
    __shared__ int s_item;
    const unsigned total = (unsigned)a.n_templates * (unsigned)F::ITEMS2;
    unsigned next = 0;
    if (threadIdx.x == 0) next = atomicAdd(a.p2_next, 1u);
    for (;;) {
        if (threadIdx.x == 0) {
            const unsigned cur = next;
            int item = -1;
            if (cur < total) {
                next = atomicAdd(a.p2_next, 1u);     // claim one ahead: its latency hides behind this item
                const long long t0 = clock64();
                if (wait_counter(a.p1_done + cur / (unsigned)F::ITEMS2, (unsigned)F::NTILES, a.abort_flag)) item = (int)cur;
                st_wait += (unsigned long long)(clock64() - t0);
            }
            s_item = item;
        }
        __syncthreads();
        const int item = s_item;
        if (item < 0) break;
        fused_p2_item<L1, L2>(a, item / F::ITEMS2, item % F::ITEMS2, smem);
        ++n_steps;
        __syncthreads();                             // s_item and the row buffers are reused
    }
}

// ---------------------------------------------------------------------------------------- kernel
template <int L1, int L2>
__global__ void __launch_bounds__(256, 2) bank_kernel(const FusedArgs a)
{
    extern __shared__ __align__(16) c2 smem[];
    using F = FusedCfg<L1, L2>;
    __shared__ int s_tile;
    const long long t_begin = clock64();
    if (threadIdx.x == 0) {
        // the first block to arrive on an SM takes a column tile (while there are tiles): one P1 block per SM
        int tile = -1;
        if (atomicAdd(a.sm_slot + smid(), 1u) == 0u) {
            const unsigned tn = atomicAdd(a.tile_next, 1u);
            if (tn < (unsigned)F::NTILES) tile = (int)tn;
        }
        s_tile = tile;
    }
    __syncthreads();
    const int tile = s_tile;
    unsigned long long st_wait = 0, n_steps = 0;
    if (tile >= 0) fused_p1_role<L1, L2>(a, tile, smem, st_wait, n_steps);
    else fused_p2_role<L1, L2>(a, smem, st_wait, n_steps);
    if (a.stats != nullptr && threadIdx.x == 0) {
        unsigned long long* o = a.stats + 6 * (size_t)blockIdx.x;
        const unsigned long long total = (unsigned long long)(clock64() - t_begin);
        o[0] = tile >= 0 ? 1ULL : 2ULL; o[1] = st_wait; o[2] = total - st_wait; o[3] = n_steps; o[4] = total;
        o[5] = (unsigned long long)(long long)tile;
    }
}

}  // namespace cbmf
