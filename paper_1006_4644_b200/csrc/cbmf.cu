// cbmf.cu -- host side of the C ABI declared in include/cbmf.h.
//
// Argument checks, device allocations and kernel launches only: every arithmetic step of
// the path (PSD tables, forward FFT of the segment, template constants, SPA generation,
// correlation, inverse FFT, |z|/sigma, arg-max, threshold, trigger sort) runs in the kernels
// of kernels.cuh.  There is no CPU fallback and nothing here touches oracle/.
#include "../../include/cbmf.h"
#include "kernels.cuh"
#include "td.cuh"
#include "cluster.h"
#include "probe.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <mutex>
#include <new>
#include <unordered_set>
#include <vector>

using namespace cbmf;

#define CBMF_MAX_STREAMS 8

struct cbmf_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int64_t n = 0;
    int log2n = 0, lg1 = 0, lg2 = 0;      // N = N1 * N2, N1 = 2^lg1 (pass 1), N2 = 2^lg2 (pass 2)
    int ifft_lg1 = 0, ifft_lg2 = 0;       // the split of the stand-alone transform (cbmf_debug_ifft)
    double fs = 0, f_low = 0, df = 0, dt = 0;
    int k_lo = 0;
    bool have_psd = false, have_seg = false;
    int pn_half_order = 4;                 // phase order of the templates: 4 = 2PN, 5 = 2.5PN (cbmf_set_pn_order)
    int sub_batch = 0;                     // templates per pass-1/pass-2 launch pair
    int max_sub_batch = 0;
    int n_streams = 1;                     // launch pairs in flight (each on its own stream and Y slice)
    int max_streams = 0;                   // slices allocated in d_Y / d_cand / d_done
    cudaStream_t aux[CBMF_MAX_STREAMS] = {};
    cudaEvent_t ev_fork = nullptr, ev_join[CBMF_MAX_STREAMS] = {};

    double* d_wfac = nullptr;              // [N/2]
    double* d_term = nullptr;              // [N/2]
    double* d_prefix = nullptr;            // [N/2]
    double* d_bsum = nullptr;              // [ceil(N/2 / SCAN_TILE)] scan block totals / offsets
    double* d_u = nullptr;                 // [N/2] k^{-1/3}
    double* d_lnk = nullptr;               // [N/2] ln k, built on the first cbmf_set_pn_order(5)
    c2* d_w = nullptr;                     // [N/2]
    c2* d_Y = nullptr;                     // [slots][N]
    c2* d_cand = nullptr;                  // [slots][N / E2] arg-max candidates, one per (row, thread)
    unsigned long long* d_key = nullptr;   // [slots] running arg-max keys
    unsigned int* d_done = nullptr;        // [max_sub_batch]
    int* d_err = nullptr;                  // [1]
    unsigned long long* d_cursor = nullptr;// [1]
    TemplCoef* d_coef = nullptr;  int64_t coef_cap = 0;
    double* d_bank = nullptr;     int64_t bank_cap = 0;
    PeakOut* d_peaks = nullptr;   int64_t peaks_cap = 0;
    TrigOut* d_trig = nullptr;    int64_t trig_cap = 0;       // entries (power of two)
    void* d_scratch = nullptr;    size_t scratch_bytes = 0;   // debug paths / load_segment

    int n_sm = 0;                          // SMs of this context's device
    // kernels whose dynamic shared-memory opt-in has been set on THIS device (cudaFuncSetAttribute is per
    // device, so the cache belongs to the context, not to the process)
    std::unordered_set<const void*> attr_set;
    unsigned int* d_tcount = nullptr;  int64_t tcount_cap = 0;    // [n_templates] triggers per template
    int* d_perr = nullptr;                 // status block + 16: set_psd found an entry <= 0 or NaN inside the band
    int* d_serr = nullptr;                 // status block + 20: load_segment found a NaN / Inf sample
    bool pend_psd = false, pend_seg = false;   // a *_dev call enqueued the check; the next waiting call resolves it
    long long* d_bad = nullptr;            // = d_cursor + 1: index of the first invalid template of the last bank, or NO_BAD_TEMPLATE
    unsigned char* h_stage = nullptr;  size_t stage_bytes = 0;    // pinned staging of a bank call's results
    int64_t last_bad = -1;

    // clustered bank call (cbmf_filter_bank_clustered): per launch pair a device trigger region and cursor, copied
    // to a ring of pinned host slots while later pairs run
    TemplCoef* d_segcoef = nullptr;        // [1] band constants of the load_segment epilogue
    int after_enqueue = 0;                 // cbmf_filter_stream: call after_enqueue_fn once the bank's launches are enqueued
    int64_t after_enqueue_seg = 0;
    int (*after_enqueue_fn)(void*, int64_t) = nullptr;
    void* after_enqueue_arg = nullptr;
    // segment streaming (cbmf_filter_stream): second weight buffer, staging and scratch of the loader stream
    c2* d_w2 = nullptr;                    // [N/2]
    c2* d_segY = nullptr;                  // [N]
    float* d_segin = nullptr;              // [N]
    int* d_segerr = nullptr;               // [1]
    cudaStream_t seg_stream = nullptr;
    cudaEvent_t ev_seg_ready[2] = {};
    TrigOut* d_ptrig = nullptr;            // [CBMF_MAX_STREAMS][PAIR_TRIG_CAP]
    unsigned long long* d_pcursor = nullptr;   // [CBMF_MAX_STREAMS]
    TrigOut* h_ptrig = nullptr;            // pinned [PIPE_RING][PAIR_TRIG_CAP]
    unsigned long long* h_pcursor = nullptr;   // pinned [PIPE_RING]
    cudaEvent_t ev_pipe[32] = {};

    // time-domain template path (cbmf_filter_bank_td)
    TdCoef* d_td = nullptr;        int64_t td_cap = 0;
    double* d_tdnorm = nullptr;    int64_t tdnorm_cap = 0;      // [n][2]
    float2* d_tdinv = nullptr;     int64_t tdinv_cap = 0;       // [n] 1/sigma_+, 1/sigma_x
    float* d_winv = nullptr;       // [N/2] 4 df / S_n
    c2* d_wd = nullptr;            // [N/2] 4 df d~ / S_n
    c2* d_tdU = nullptr;           int64_t tdU_cap = 0;         // [templates per step][N]

    int64_t launches = 0;
    int profiling = 0;                     // 0 off, 1 every launch alone on the context's stream, 2 in the real schedule
    std::vector<cudaEvent_t> ev[2];        // per pass: start/stop pairs of the last filter call
    size_t ev_used[2] = {0, 0};
    std::vector<float> timeline[2];        // per pass: (start, end) in ms of every launch of the last profiled call
    double last_ms[2] = {0, 0};
    int64_t last_launches[2] = {0, 0};
    char cuda_err[256] = {0};
};

namespace {

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; }
        if (prev != dev) ok = (cudaSetDevice(dev) == cudaSuccess);
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int cuda_fail(cbmf_ctx* c, cudaError_t e, const char* what)
{
    if (c) snprintf(c->cuda_err, sizeof(c->cuda_err), "%s: %s", what, cudaGetErrorString(e));
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? CBMF_ENOMEM : CBMF_ECUDA;
}
#define CU(call)                                                         \
    do {                                                                 \
        cudaError_t e__ = (call);                                        \
        if (e__ != cudaSuccess) return cuda_fail(c, e__, #call);         \
    } while (0)

template <typename T>
int grow(cbmf_ctx* c, T*& p, int64_t& cap, int64_t need)
{
    if (need <= cap) return CBMF_OK;
    if (p) { CU(cudaFree(p)); p = nullptr; cap = 0; }
    CU(cudaMalloc(&p, sizeof(T) * (size_t)need));
    cap = need;
    return CBMF_OK;
}

int grow_scratch(cbmf_ctx* c, size_t bytes)
{
    if (bytes <= c->scratch_bytes) return CBMF_OK;
    if (c->d_scratch) { CU(cudaFree(c->d_scratch)); c->d_scratch = nullptr; c->scratch_bytes = 0; }
    CU(cudaMalloc(&c->d_scratch, bytes));
    c->scratch_bytes = bytes;
    return CBMF_OK;
}

int ilog2(int64_t n) { int l = 0; while ((int64_t(1) << l) < n) ++l; return l; }

// ---------------------------------------------------------------- launch dispatch over (N1, N2)
// Blocks per column tile of a pass-1 launch (LOAD_GEN).  Each block stages its tile of w once and walks
// through its share of the templates, so FEW, LONG-LIVED blocks are wanted (+12 % over
// short-lived blocks at 4 streams): as many as the SMs hold at once, two per SM.  With four launch pairs in
// flight the block scheduler then mixes them with the pass-2 blocks of the other pairs on every SM, which
// pairs the generator / exchange phases of pass 1 with the FMA-bound row FFTs of pass 2; a launch timed alone
// fills the GPU by itself (one block per SM left half of every SM idle in that measurement, same bank throughput).
// Series for k^{-1/3} in the generator (spa_correlate): valid where (columns of a tile - 1) / (first bin
// of the first in-band row) <= 2e-3.
bool p1_series_ok(int k_lo, int l2, int tile_cols)
{
    const int k1_lo = k_lo / l2;
    return k1_lo >= 1 && (double)(tile_cols - 1) <= 2e-3 * (double)k1_lo * (double)l2;
}

int p1_groups(int n_sm, int n_tiles, int batch)
{
    int g = 2 * n_sm / n_tiles;            // two blocks fit an SM (registers, shared memory)
    if (g < 1) g = 1;
    if (g > batch) g = batch;
    return g;
}

// Opt a kernel in to `bytes` of dynamic shared memory on the context's device, once per context.
template <typename K>
cudaError_t ensure_smem_attr(cbmf_ctx* c, K kernel, size_t bytes)
{
    const void* key = reinterpret_cast<const void*>(kernel);
    if (c->attr_set.count(key)) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) c->attr_set.insert(key);
    return e;
}

template <int L1, int L2, int MODE>
cudaError_t launch_p1_L(cbmf_ctx* c, cudaStream_t s, P1Args a, int batch)
{
    const size_t smem = p1_smem_bytes<L1, MODE>();
    cudaError_t e = ensure_smem_attr(c, p1_kernel<L1, L2, MODE>, smem);
    if (e != cudaSuccess) return e;
    a.batch = batch;
    constexpr bool GEN = (MODE == LOAD_GEN || MODE == LOAD_GEN_DUMP);
    if (GEN) {
        // expansion about the first column of a tile (spa_generate_rows, spa_correlate): valid where
        // (columns of a tile - 1) / (first in-band bin of a row) <= 2e-3
        a.use_series = p1_series_ok(a.use_series, L2, Cfg<L1>::C) ? 1 : 0;    // the caller passes k_lo in use_series
    }
    const int groups = GEN ? p1_groups(c->n_sm, L2 / Cfg<L1>::C, batch) : batch;
    dim3 grid(L2 / Cfg<L1>::C, groups);
    p1_kernel<L1, L2, MODE><<<grid, Cfg<L1>::NT1, smem, s>>>(a);
    return cudaGetLastError();
}

template <int L1, int L2, int MODE>
constexpr int p2_items() { return L1 / (Cfg<L2>::ROWS * (MODE == EPI_MAX ? p2_rpw<L1, L2>() : 1)); }

template <int L1, int L2, int MODE, bool MASK = false>
cudaError_t launch_p2_L(cbmf_ctx* c, cudaStream_t s, const P2Args& a, int batch)
{
    const size_t smem = sizeof(c2) * (size_t)p2_row_stride<L2>() * Cfg<L2>::ROWS;
    cudaError_t e = ensure_smem_attr(c, p2_kernel<L1, L2, MODE, MASK>, smem);
    if (e != cudaSuccess) return e;
    dim3 grid(p2_items<L1, L2, MODE>(), batch);
    p2_kernel<L1, L2, MODE, MASK><<<grid, Cfg<L2>::NT2, smem, s>>>(a);
    return cudaGetLastError();
}

// N = 2^(lg1 + lg2), 6 <= lg1, lg2 <= 12: the splits cbmf_create chooses
#define CBMF_DISPATCH(lg1, lg2, EXPR)                                               \
    switch ((lg1) * 32 + (lg2)) {                                                  \
        case 6 * 32 + 6:   { constexpr int L1 = 64,   L2 = 64;   return EXPR; }    \
        case 6 * 32 + 7:   { constexpr int L1 = 64,   L2 = 128;  return EXPR; }    \
        case 7 * 32 + 7:   { constexpr int L1 = 128,  L2 = 128;  return EXPR; }    \
        case 7 * 32 + 8:   { constexpr int L1 = 128,  L2 = 256;  return EXPR; }    \
        case 8 * 32 + 8:   { constexpr int L1 = 256,  L2 = 256;  return EXPR; }    \
        case 8 * 32 + 9:   { constexpr int L1 = 256,  L2 = 512;  return EXPR; }    \
        case 9 * 32 + 9:   { constexpr int L1 = 512,  L2 = 512;  return EXPR; }    \
        case 9 * 32 + 10:  { constexpr int L1 = 512,  L2 = 1024; return EXPR; }    \
        case 10 * 32 + 10: { constexpr int L1 = 1024, L2 = 1024; return EXPR; }    \
        case 11 * 32 + 10: { constexpr int L1 = 2048, L2 = 1024; return EXPR; }    \
        case 12 * 32 + 10: { constexpr int L1 = 4096, L2 = 1024; return EXPR; }    \
        case 11 * 32 + 12: { constexpr int L1 = 2048, L2 = 4096; return EXPR; }    \
        case 12 * 32 + 12: { constexpr int L1 = 4096, L2 = 4096; return EXPR; }    \
        default: return cudaErrorInvalidValue;                                      \
    }

template <int MODE>
cudaError_t launch_p1(cbmf_ctx* c, cudaStream_t s, const P1Args& a, int batch)
{
    CBMF_DISPATCH(c->lg1, c->lg2, (launch_p1_L<L1, L2, MODE>(c, s, a, batch)))
}
template <int MODE, bool MASK = false>
cudaError_t launch_p2(cbmf_ctx* c, cudaStream_t s, const P2Args& a, int batch)
{
    CBMF_DISPATCH(c->lg1, c->lg2, (launch_p2_L<L1, L2, MODE, MASK>(c, s, a, batch)))
}

// The stand-alone transform (plain load and store epilogues only) with its own split.
cudaError_t launch_p1_ifft(cbmf_ctx* c, cudaStream_t s, const P1Args& a, int batch)
{
    if (c->ifft_lg1 == 10 && c->ifft_lg2 == 11) return launch_p1_L<1024, 2048, LOAD_CPLX>(c, s, a, batch);
    if (c->ifft_lg1 == 11 && c->ifft_lg2 == 11) return launch_p1_L<2048, 2048, LOAD_CPLX>(c, s, a, batch);
    return launch_p1<LOAD_CPLX>(c, s, a, batch);
}
cudaError_t launch_p2_ifft(cbmf_ctx* c, cudaStream_t s, const P2Args& a, int batch)
{
    if (c->ifft_lg1 == 10 && c->ifft_lg2 == 11) return launch_p2_L<1024, 2048, EPI_STORE>(c, s, a, batch);
    if (c->ifft_lg1 == 11 && c->ifft_lg2 == 11) return launch_p2_L<2048, 2048, EPI_STORE>(c, s, a, batch);
    return launch_p2<EPI_STORE>(c, s, a, batch);
}

// candidate slots per template of the arg-max pass: one per (row j1, thread of the row group) = N / E2
template <int L1, int L2> constexpr int cand_count() { return L1 * Cfg<L2>::T; }
size_t cand_per_template(const cbmf_ctx* c)
{
    auto f = [&]() -> int { CBMF_DISPATCH(c->lg1, c->lg2, (cand_count<L1, L2>())) };
    const int v = f();
    return v > 0 ? (size_t)v : 1;
}

// pass-timing events (cbmf_set_profiling): one start/stop pair per launch
int ev_begin(cbmf_ctx* c, int which, cudaStream_t st)
{
    if (!c->profiling) return CBMF_OK;
    auto& v = c->ev[which];
    if (c->ev_used[which] + 2 > v.size()) {
        for (int i = 0; i < 2; ++i) { cudaEvent_t e; CU(cudaEventCreate(&e)); v.push_back(e); }
    }
    CU(cudaEventRecord(v[c->ev_used[which]], st));
    return CBMF_OK;
}
int ev_end(cbmf_ctx* c, int which, cudaStream_t st)
{
    if (!c->profiling) return CBMF_OK;
    CU(cudaEventRecord(c->ev[which][c->ev_used[which] + 1], st));
    c->ev_used[which] += 2;
    return CBMF_OK;
}
int ev_collect(cbmf_ctx* c)
{
    for (int w = 0; w < 2; ++w) {
        c->last_ms[w] = 0; c->last_launches[w] = 0;
        if (!c->profiling) continue;
        c->timeline[w].clear();
        for (size_t i = 0; i + 1 < c->ev_used[w]; i += 2) {
            float ms = 0.f, t0 = 0.f;
            CU(cudaEventElapsedTime(&ms, c->ev[w][i], c->ev[w][i + 1]));
            c->last_ms[w] += ms; c->last_launches[w] += 1;
            if (c->ev_used[0] >= 2) CU(cudaEventElapsedTime(&t0, c->ev[0][0], c->ev[w][i]));    // since the first pass-1 launch
            c->timeline[w].push_back(t0);
            c->timeline[w].push_back(t0 + ms);
        }
    }
    return CBMF_OK;
}

// (Re)allocate the per-slot buffers for `sb` templates per launch pair and `ns` pairs in flight.
int alloc_pipeline(cbmf_ctx* c, int sb, int ns)
{
    if (sb <= c->max_sub_batch && ns <= c->max_streams) return CBMF_OK;
    if (sb < c->max_sub_batch) sb = c->max_sub_batch;
    if (ns < c->max_streams) ns = c->max_streams;
    CU(cudaStreamSynchronize(c->stream));
    for (int i = 0; i < c->max_streams; ++i) if (c->aux[i]) CU(cudaStreamSynchronize(c->aux[i]));
    const size_t slots = (size_t)sb * ns;
    const size_t ncand = cand_per_template(c);
    c2* y = nullptr; c2* cand = nullptr; unsigned int* done = nullptr; unsigned long long* key = nullptr;
    cudaError_t e = cudaMalloc(&y, sizeof(c2) * (size_t)c->n * slots);
    if (e == cudaSuccess) e = cudaMalloc(&cand, sizeof(c2) * ncand * slots);
    if (e == cudaSuccess) e = cudaMalloc(&done, sizeof(unsigned int) * slots);
    if (e == cudaSuccess) e = cudaMalloc(&key, sizeof(unsigned long long) * slots);
    if (e == cudaSuccess) e = cudaMemsetAsync(done, 0, sizeof(unsigned int) * slots, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(key, 0, sizeof(unsigned long long) * slots, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    for (int i = c->max_streams; i < ns && e == cudaSuccess; ++i) {
        e = cudaStreamCreateWithFlags(&c->aux[i], cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_join[i], cudaEventDisableTiming);
    }
    if (e == cudaSuccess && !c->ev_fork) e = cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming);
    if (e != cudaSuccess) { cudaFree(y); cudaFree(cand); cudaFree(done); cudaFree(key); return cuda_fail(c, e, "alloc_pipeline"); }
    cudaFree(c->d_Y); cudaFree(c->d_cand); cudaFree(c->d_done); cudaFree(c->d_key);
    c->d_Y = y; c->d_cand = cand; c->d_done = done; c->d_key = key;
    c->max_sub_batch = sb; c->max_streams = ns;
    return CBMF_OK;
}

}  // namespace

// ======================================================================= create / destroy
extern "C" int cbmf_destroy(cbmf_ctx* c)
{
    if (!c) return CBMF_EINVAL;
    DeviceGuard g(c->device);
    cudaStreamSynchronize(c->stream);
    cudaFree(c->d_wfac); cudaFree(c->d_term); cudaFree(c->d_prefix); cudaFree(c->d_bsum); cudaFree(c->d_w);
    cudaFree(c->d_Y); cudaFree(c->d_cand); cudaFree(c->d_done); cudaFree(c->d_key); cudaFree(c->d_err); cudaFree(c->d_u);
    cudaFree(c->d_lnk); cudaFree(c->d_cursor); cudaFree(c->d_coef); cudaFree(c->d_bank); cudaFree(c->d_peaks);
    cudaFree(c->d_trig); cudaFree(c->d_scratch); cudaFree(c->d_tcount); cudaFreeHost(c->h_stage);
    cudaFree(c->d_segcoef); cudaFree(c->d_w2); cudaFree(c->d_segY); cudaFree(c->d_segin); cudaFree(c->d_segerr);
    if (c->seg_stream) { cudaStreamSynchronize(c->seg_stream); cudaStreamDestroy(c->seg_stream); }
    for (cudaEvent_t e : c->ev_seg_ready) if (e) cudaEventDestroy(e);
    cudaFree(c->d_ptrig); cudaFree(c->d_pcursor); cudaFreeHost(c->h_ptrig); cudaFreeHost(c->h_pcursor);
    cudaFree(c->d_td); cudaFree(c->d_tdnorm); cudaFree(c->d_tdinv); cudaFree(c->d_winv); cudaFree(c->d_wd); cudaFree(c->d_tdU);
    for (cudaEvent_t e : c->ev_pipe) if (e) cudaEventDestroy(e);
    for (int w = 0; w < 2; ++w) for (cudaEvent_t e : c->ev[w]) cudaEventDestroy(e);
    for (int i = 0; i < CBMF_MAX_STREAMS; ++i) {
        if (c->aux[i]) { cudaStreamSynchronize(c->aux[i]); cudaStreamDestroy(c->aux[i]); }
        if (c->ev_join[i]) cudaEventDestroy(c->ev_join[i]);
    }
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    cudaGetLastError();
    delete c;
    return CBMF_OK;
}

extern "C" int cbmf_create(cbmf_ctx** out, int device, int64_t n, double fs_hz, double f_low_hz,
                           void* cuda_stream)
{
    if (!out) return CBMF_EINVAL;
    *out = nullptr;
    // 2^12 <= n: the two-pass split needs N1, N2 >= 64 (DESIGN.md §3 records the floor against SURVEY.md §8(b)'s 2^10)
    if (n < (int64_t(1) << 12) || n > (int64_t(1) << 24) || (n & (n - 1)) != 0) return CBMF_EINVAL;
    if (!(fs_hz > 0) || !std::isfinite(fs_hz)) return CBMF_EINVAL;
    if (!(f_low_hz > 0) || !(f_low_hz < 0.5 * fs_hz)) return CBMF_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess) { cudaGetLastError(); return CBMF_ECUDA; }
    if (device < 0 || device >= ndev) return CBMF_EINVAL;

    cbmf_ctx* c = new (std::nothrow) cbmf_ctx();
    if (!c) return CBMF_ENOMEM;
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    c->n = n;
    c->log2n = ilog2(n);
    c->lg1 = c->log2n / 2;                 // the longer FFT goes to pass 2 (contiguous rows) ...
    c->lg2 = c->log2n - c->lg1;
    // ... except at N = 2^21 and 2^22, where pass 2 keeps its best shape (rows of 1024 points, one warp per row,
    // one exchange) and pass 1 takes the 2048- / 4096-point columns: 22 % / 34 % faster than 1024 x 2048 / 2048 x 2048
    if (c->log2n == 21 || c->log2n == 22) { c->lg2 = 10; c->lg1 = c->log2n - 10; }
    // the stand-alone transform (cbmf_debug_ifft: all N inputs non-zero, plain store epilogue) prefers the shorter
    // column FFT at these sizes: 1024 x 2048 and 2048 x 2048 run at 0.97-0.99 of the library transform, against 0.75
    c->ifft_lg1 = c->lg1; c->ifft_lg2 = c->lg2;
    if (c->log2n == 21) { c->ifft_lg1 = 10; c->ifft_lg2 = 11; }
    if (c->log2n == 22) { c->ifft_lg1 = 11; c->ifft_lg2 = 11; }
    c->fs = fs_hz; c->f_low = f_low_hz;
    c->df = fs_hz / (double)n; c->dt = 1.0 / fs_hz;
    c->k_lo = (int)std::ceil(f_low_hz * ((double)n / fs_hz));       // reading A7: inclusive, in double
    if (c->k_lo < 1) c->k_lo = 1;

    // templates per launch pair: up to 2 GiB of inter-pass buffer per pair (256 templates at N = 2^20).  Measured
    // (DESIGN.md §7): long launches matter more than keeping Y inside the L2 at the present kernel speed
    // (cfg2: 282 k templates/s at 64 per pair, 286 k at 128, 288 k at 256).  A call uses fewer per pair when the
    // bank is too small to give every stream a pair (eff_sub_batch).
    int64_t sb = (int64_t(2048) << 20) / (8 * n);
    if (sb < 1) sb = 1;
    if (sb > 256) sb = 256;
    const int ns = 4;                      // launch pairs in flight (cbmf_set_streams)
    c->sub_batch = (int)sb;
    c->n_streams = ns;

    DeviceGuard g(device);
    auto fail = [&](int rc) { cbmf_destroy(c); return rc; };
    if (!g.ok) return fail(CBMF_ECUDA);
    const size_t nh = (size_t)n / 2;
#define CUF(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return fail(cuda_fail(nullptr, e__, #call)); } while (0)
    CUF(cudaMalloc(&c->d_wfac, sizeof(double) * nh));
    CUF(cudaMalloc(&c->d_term, sizeof(double) * nh));
    CUF(cudaMalloc(&c->d_prefix, sizeof(double) * nh));
    CUF(cudaMalloc(&c->d_bsum, sizeof(double) * ((nh + SCAN_TILE - 1) / SCAN_TILE)));
    CUF(cudaMalloc(&c->d_w, sizeof(c2) * nh));
    CUF(cudaMalloc(&c->d_u, sizeof(double) * nh));
    CUF(cudaMalloc(&c->d_err, sizeof(int)));
    // status block of a bank call: {trigger cursor, first invalid template}: one reset copy, one read-back
    CUF(cudaMalloc(&c->d_cursor, 4 * sizeof(unsigned long long)));
    CUF(cudaMemset(c->d_cursor, 0, 4 * sizeof(unsigned long long)));
    c->d_bad = reinterpret_cast<long long*>(c->d_cursor + 1);
    c->d_perr = reinterpret_cast<int*>(c->d_cursor + 2);
    c->d_serr = c->d_perr + 1;
    CUF(cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, device));
    CUF(cudaMemsetAsync(c->d_err, 0, sizeof(int), c->stream));
    rcbrt_table_kernel<<<(unsigned)((nh + 255) / 256), 256, 0, c->stream>>>(c->d_u, (int)nh);
    CUF(cudaGetLastError());
    c->launches += 1;
    CUF(cudaStreamSynchronize(c->stream));
#undef CUF
    { const int rc = alloc_pipeline(c, c->sub_batch, c->n_streams); if (rc) return fail(rc); }
    *out = c;
    return CBMF_OK;
}

extern "C" int cbmf_set_sub_batch(cbmf_ctx* c, int templates_per_launch)
{
    if (!c || templates_per_launch < 1 || templates_per_launch > 4096) return CBMF_EINVAL;
    DeviceGuard g(c->device);
    const int rc = alloc_pipeline(c, templates_per_launch, c->n_streams);
    if (rc) return rc;
    c->sub_batch = templates_per_launch;
    return CBMF_OK;
}

extern "C" int cbmf_set_streams(cbmf_ctx* c, int launch_pairs_in_flight)
{
    if (!c || launch_pairs_in_flight < 1 || launch_pairs_in_flight > CBMF_MAX_STREAMS) return CBMF_EINVAL;
    DeviceGuard g(c->device);
    const int rc = alloc_pipeline(c, c->sub_batch, launch_pairs_in_flight);
    if (rc) return rc;
    c->n_streams = launch_pairs_in_flight;
    return CBMF_OK;
}

extern "C" int cbmf_get_streams(const cbmf_ctx* c) { return c ? c->n_streams : CBMF_EINVAL; }

extern "C" int cbmf_get_sub_batch(const cbmf_ctx* c) { return c ? c->sub_batch : CBMF_EINVAL; }

extern "C" int cbmf_set_pn_order(cbmf_ctx* c, int half_order)
{
    if (!c || (half_order != 4 && half_order != 5)) return CBMF_EINVAL;
    if (half_order == 5 && !c->d_lnk) {
        DeviceGuard g(c->device);
        const size_t nh = (size_t)c->n / 2;
        CU(cudaMalloc(&c->d_lnk, sizeof(double) * nh));
        lnk_table_kernel<<<(unsigned)((nh + 255) / 256), 256, 0, c->stream>>>(c->d_lnk, (int)nh);
        CU(cudaGetLastError());
        c->launches += 1;
        CU(cudaStreamSynchronize(c->stream));
    }
    c->pn_half_order = half_order;
    return CBMF_OK;
}
extern "C" int cbmf_get_pn_order(const cbmf_ctx* c) { return c ? c->pn_half_order : CBMF_EINVAL; }

extern "C" int cbmf_get_split(const cbmf_ctx* c, int* log2_n1, int* log2_n2)
{
    if (!c) return CBMF_EINVAL;
    if (log2_n1) *log2_n1 = c->lg1;
    if (log2_n2) *log2_n2 = c->lg2;
    return CBMF_OK;
}

extern "C" int64_t cbmf_last_bad_template(const cbmf_ctx* c) { return c ? c->last_bad : -1; }

// ======================================================================= S0: set_psd
// Resolve the input checks that the *_dev calls enqueue without waiting (cbmf.h): one 8-byte read-back.
static int check_pending(cbmf_ctx* c)
{
    if (!c->pend_psd && !c->pend_seg) return CBMF_OK;
    int err[2] = {0, 0};
    CU(cudaMemcpyAsync(err, c->d_perr, sizeof(err), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    const bool bad_psd = c->pend_psd && err[0], bad_seg = c->pend_seg && err[1];
    c->pend_psd = c->pend_seg = false;
    if (bad_psd) { c->have_psd = false; c->have_seg = false; return CBMF_EINVAL; }
    if (bad_seg) { c->have_seg = false; return CBMF_EINVAL; }
    return CBMF_OK;
}

// defer: enqueue only and report an invalid entry at the next call that waits (the *_dev entry point).
static int set_psd_impl(cbmf_ctx* c, const double* psd_dev, bool defer)
{
    const int nh = (int)(c->n / 2);
    c->have_psd = false; c->have_seg = false;
    c->pend_psd = c->pend_seg = false;
    CU(cudaMemsetAsync(c->d_perr, 0, 2 * sizeof(int), c->stream));
    const int nblk = (nh + SCAN_TILE - 1) / SCAN_TILE;
    psd_terms_kernel<<<nblk, SCAN_THREADS, 0, c->stream>>>(psd_dev, c->d_wfac, c->d_term, c->d_bsum, nh, c->k_lo,
                                                           c->df, c->dt, c->d_perr);
    CU(cudaGetLastError());
    scan_block_sums_kernel<<<1, SCAN_THREADS, 0, c->stream>>>(c->d_bsum, nblk);
    CU(cudaGetLastError());
    prefix_tile_kernel<<<nblk, SCAN_THREADS, 0, c->stream>>>(c->d_term, c->d_bsum, c->d_prefix, nh);
    CU(cudaGetLastError());
    c->launches += 3;
    c->have_psd = true;
    c->pend_psd = true;
    return defer ? CBMF_OK : check_pending(c);
}

extern "C" int cbmf_set_psd_dev(cbmf_ctx* c, const double* psd_dev, int64_t n_bins)
{
    if (!c || !psd_dev) return CBMF_EINVAL;
    if (n_bins != c->n / 2 + 1) return CBMF_EINVAL;
    DeviceGuard g(c->device);
    return set_psd_impl(c, psd_dev, true);
}

extern "C" int cbmf_set_psd(cbmf_ctx* c, const double* psd, int64_t n_bins)
{
    if (!c || !psd) return CBMF_EINVAL;
    if (n_bins != c->n / 2 + 1) return CBMF_EINVAL;
    DeviceGuard g(c->device);
    int rc = grow_scratch(c, sizeof(double) * (size_t)n_bins);
    if (rc) return rc;
    CU(cudaMemcpyAsync(c->d_scratch, psd, sizeof(double) * (size_t)n_bins, cudaMemcpyHostToDevice, c->stream));
    return set_psd_impl(c, (const double*)c->d_scratch, false);
}

// ======================================================================= S1: load_segment
// d~[k] = dt conj(IDFT(d)[k]) for real d, so the forward transform reuses the inverse kernels.
// Enqueue only: samples_dev -> w_out on stream st, with Y_scratch (n complex) as the inter-pass buffer and *err_flag
// set on a non-finite sample.
static int enqueue_load_segment(cbmf_ctx* c, const float* samples_dev, c2* w_out, c2* Y_scratch, cudaStream_t st, int* err_flag)
{
    // k_lo travels to the EPI_WSTORE epilogue in a one-entry TemplCoef of its own (a bank may be reading d_coef)
    if (!c->d_segcoef) {
        CU(cudaMalloc(&c->d_segcoef, sizeof(TemplCoef)));
        TemplCoef tc; memset(&tc, 0, sizeof(tc)); tc.k_lo = c->k_lo; tc.k_hi = (int)(c->n / 2 - 1);
        CU(cudaMemcpy(c->d_segcoef, &tc, sizeof(tc), cudaMemcpyHostToDevice));
    }
    CU(cudaMemsetAsync(err_flag, 0, sizeof(int), st));
    P1Args a1; memset(&a1, 0, sizeof(a1));
    a1.in_r = samples_dev; a1.Y = Y_scratch; a1.err_flag = err_flag;
    CU(launch_p1<LOAD_REAL>(c, st, a1, 1));
    P2Args a2; memset(&a2, 0, sizeof(a2));
    a2.Y = Y_scratch; a2.coef = c->d_segcoef; a2.w_out = w_out; a2.wfac = c->d_wfac;
    CU(launch_p2<EPI_WSTORE>(c, st, a2, 1));
    c->launches += 2;
    return CBMF_OK;
}

static int load_segment_impl(cbmf_ctx* c, const float* samples_dev, bool defer)
{
    c->have_seg = false;
    int rc = enqueue_load_segment(c, samples_dev, c->d_w, c->d_Y, c->stream, c->d_serr);
    if (rc) return rc;
    c->have_seg = true;
    c->pend_seg = true;
    return defer ? CBMF_OK : check_pending(c);
}

extern "C" int cbmf_load_segment_dev(cbmf_ctx* c, const float* samples_dev, int64_t n_samples)
{
    if (!c || !samples_dev) return CBMF_EINVAL;
    if (n_samples != c->n) return CBMF_EINVAL;
    if (!c->have_psd) return CBMF_ESTATE;
    DeviceGuard g(c->device);
    return load_segment_impl(c, samples_dev, true);
}

extern "C" int cbmf_load_segment(cbmf_ctx* c, const float* samples, int64_t n_samples)
{
    if (!c || !samples) return CBMF_EINVAL;
    if (n_samples != c->n) return CBMF_EINVAL;
    if (!c->have_psd) return CBMF_ESTATE;
    DeviceGuard g(c->device);
    int rc = check_pending(c);
    if (rc) return rc;
    if ((rc = grow_scratch(c, sizeof(float) * (size_t)c->n))) return rc;
    CU(cudaMemcpyAsync(c->d_scratch, samples, sizeof(float) * (size_t)c->n, cudaMemcpyHostToDevice, c->stream));
    return load_segment_impl(c, (const float*)c->d_scratch, false);
}

// ======================================================================= S2-S8: filter_bank
// Sort the first `count` entries of c->d_trig by (template, sample) on the device.
static int sort_triggers(cbmf_ctx* c, int64_t count)
{
    if (count <= 1) return CBMF_OK;
    long long np2 = 1;
    while (np2 < count) np2 <<= 1;
    if (np2 <= TRIG_SMALL) {
        const size_t smem_small = (sizeof(unsigned long long) + sizeof(TrigOut) + sizeof(unsigned short)) * (size_t)np2;
        CU(ensure_smem_attr(c, trig_sort_small_kernel,
                            (sizeof(unsigned long long) + sizeof(TrigOut) + sizeof(unsigned short)) * TRIG_SMALL));
        trig_sort_small_kernel<<<1, 1024, smem_small, c->stream>>>(c->d_trig, (int)count, (int)np2);
        CU(cudaGetLastError());
        c->launches += 1;
        return CBMF_OK;
    }
    const int tile = (int)(np2 < TRIG_TILE ? np2 : TRIG_TILE);
    const size_t smem = sizeof(TrigOut) * (size_t)tile;
    CU(ensure_smem_attr(c, trig_sort_tile_kernel, sizeof(TrigOut) * TRIG_TILE));
    const unsigned tiles = (unsigned)(np2 / tile);
    trig_sort_tile_kernel<<<tiles, 1024, smem, c->stream>>>(c->d_trig, count, tile, 0);
    CU(cudaGetLastError());
    c->launches += 1;
    const unsigned blocks = (unsigned)((np2 + 255) / 256);
    for (long long kk = 2LL * tile; kk <= np2; kk <<= 1) {
        for (long long jj = kk >> 1; jj >= tile; jj >>= 1) {
            trig_bitonic_kernel<<<blocks, 256, 0, c->stream>>>(c->d_trig, np2, kk, jj);
            CU(cudaGetLastError());
            c->launches += 1;
        }
        trig_sort_tile_kernel<<<tiles, 1024, smem, c->stream>>>(c->d_trig, count, tile, kk);
        CU(cudaGetLastError());
        c->launches += 1;
    }
    return CBMF_OK;
}

// Templates per launch pair of a call over nt templates: the context's sub-batch, or fewer so that every stream gets
// a pair (at least 16 where the bank has them).
static int eff_sub_batch(const cbmf_ctx* c, int64_t nt)
{
    int64_t per = (nt + c->n_streams - 1) / c->n_streams;
    const int64_t floor16 = nt < 16 ? nt : 16;
    if (per < floor16) per = floor16;
    int64_t sb = c->sub_batch < per ? c->sub_batch : per;
    return (int)(sb < 1 ? 1 : sb);
}

// Pass-1 / pass-2 launch pairs for templates [0, nt) whose constants are in c->d_coef; peaks to c->d_peaks,
// triggers to c->d_trig (dev_cap entries; the total is counted in c->d_cursor whatever the capacity).
static int run_bank_passes(cbmf_ctx* c, int64_t nt, int64_t dev_cap, const c2* w = nullptr, int j_min = 0)
{
    if (!w) w = c->d_w;
    int rc;
    const int sb = eff_sub_batch(c, nt);
    // Launch pairs go round-robin over ns streams, each with its own slice of Y / cand / done, so
    // that the tail of one kernel overlaps the head of the next pair.  With per-pass event timing on
    // (cbmf_set_profiling mode 1) everything stays on the context's stream: each launch is timed alone;
    // mode 2 keeps the real schedule and brackets every launch with events on its own stream.
    const int ns = (c->profiling == 1 || nt <= sb) ? 1 : c->n_streams;
    const size_t ncand = cand_per_template(c);
    if (ns > 1) {
        CU(cudaEventRecord(c->ev_fork, c->stream));
        for (int s = 0; s < ns; ++s) CU(cudaStreamWaitEvent(c->aux[s], c->ev_fork, 0));
    }
    int64_t pair = 0;
    for (int64_t t0 = 0; t0 < nt; t0 += sb, ++pair) {
        const int nb = (int)((nt - t0 < sb) ? (nt - t0) : sb);
        const int slot = (int)(pair % ns);
        cudaStream_t st = (ns > 1) ? c->aux[slot] : c->stream;
        c2* Y = c->d_Y + (size_t)slot * c->max_sub_batch * (size_t)c->n;
        P1Args a1; memset(&a1, 0, sizeof(a1));
        a1.w = w; a1.u = c->d_u; a1.lnk = c->d_lnk; a1.coef = c->d_coef + t0; a1.Y = Y; a1.err_flag = c->d_err; a1.use_series = c->k_lo; a1.bad = c->d_bad;
        if ((rc = ev_begin(c, 0, st))) return rc;
        CU(launch_p1<LOAD_GEN>(c, st, a1, nb));
        if ((rc = ev_end(c, 0, st))) return rc;
        P2Args a2; memset(&a2, 0, sizeof(a2));
        a2.Y = Y; a2.coef = c->d_coef + t0;
        a2.cand = c->d_cand + (size_t)slot * c->max_sub_batch * ncand;
        a2.best_key = c->d_key + (size_t)slot * c->max_sub_batch;
        a2.done_ctr = c->d_done + (size_t)slot * c->max_sub_batch; a2.peaks = c->d_peaks + t0; a2.trig = c->d_trig;
        a2.trig_cursor = c->d_cursor; a2.trig_cap = (unsigned long long)dev_cap;
        a2.trig_count = c->d_tcount + t0;
        a2.tmpl_base = (int)t0;
        a2.j_min = j_min;
        a2.bad = c->d_bad;
        if ((rc = ev_begin(c, 1, st))) return rc;
        if (j_min > 0) CU((launch_p2<EPI_MAX, true>(c, st, a2, nb)));
        else CU(launch_p2<EPI_MAX>(c, st, a2, nb));
        if ((rc = ev_end(c, 1, st))) return rc;
        c->launches += 2;
    }
    if (ns > 1) {
        for (int s = 0; s < ns; ++s) {
            CU(cudaEventRecord(c->ev_join[s], c->aux[s]));
            CU(cudaStreamWaitEvent(c->stream, c->ev_join[s], 0));
        }
    }
    if (c->after_enqueue && c->after_enqueue_fn) {
        c->after_enqueue = 0;                   // once per bank (a truncated list repeats the passes)
        if ((rc = c->after_enqueue_fn(c->after_enqueue_arg, c->after_enqueue_seg))) return rc;
    }
    return CBMF_OK;
}

// Template constants of a bank (S2) into c->d_coef, with the early check: an invalid template fails the call here,
// before any filtering, and is named (cbmf_last_bad_template).  bank_dev: [n][2] doubles on the device.
static int bank_setup(cbmf_ctx* c, const double* bank_dev, int64_t nt, float thr)
{
    int rc;
    c->last_bad = -1;
    if ((rc = grow(c, c->d_coef, c->coef_cap, nt))) return rc;
    if ((rc = grow(c, c->d_peaks, c->peaks_cap, nt))) return rc;
    if ((rc = grow(c, c->d_tcount, c->tcount_cap, nt))) return rc;
    const long long no_bad = NO_BAD_TEMPLATE;
    CU(cudaMemsetAsync(c->d_err, 0, sizeof(int), c->stream));
    CU(cudaMemcpyAsync(c->d_bad, &no_bad, sizeof(long long), cudaMemcpyHostToDevice, c->stream));
    SetupArgs sa;
    sa.tcount = nullptr;
    sa.bank = bank_dev; sa.prefix = c->d_prefix; sa.coef = c->d_coef; sa.n_templates = (int)nt;
    sa.n_half = (int)(c->n / 2); sa.k_lo = c->k_lo; sa.n_over_fs = (double)c->n / c->fs; sa.df = c->df;
    sa.threshold = thr; sa.err_flag = c->d_err; sa.bad_idx = c->d_bad; sa.pn_half_order = c->pn_half_order;
    template_setup_kernel<<<(unsigned)((nt + 127) / 128), 128, 0, c->stream>>>(sa);
    CU(cudaGetLastError());
    c->launches += 1;
    long long bad = no_bad;
    CU(cudaMemcpyAsync(&bad, c->d_bad, sizeof(long long), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (bad != no_bad) { c->last_bad = (int64_t)bad; return CBMF_EINVAL; }
    return CBMF_OK;
}

// The general trigger collection behind a bank pass over templates [0, nt) that has completed with `found` triggers
// counted (c->d_cursor) and at most c->trig_cap of them on the device: a list of any size is sorted and its first
// trig_capacity entries delivered with the peaks (host or device pointers, out_kind); a list the device buffer could
// not hold is rebuilt first.  Shared by the plain bank call, the streamed segments and the single-pair re-runs of
// the clustered call.  -> CBMF_WTRUNC if found > trig_capacity.
static int collect_triggers(cbmf_ctx* c, int64_t nt, const c2* w, int j_min, int64_t found, void* peaks_out,
                            void* trig_out, int64_t trig_capacity, cudaMemcpyKind out_kind)
{
    int rc;
    const int64_t kept = found < trig_capacity ? found : trig_capacity;
    if (kept > 0 && trig_out) {
        int64_t on_device = found;
        if (found > c->trig_cap) {
            // Truncated and the device list is incomplete.  The contract (cbmf.h) keeps the FIRST trig_capacity
            // triggers in (template, sample) order, so the whole lists of the leading templates are needed:
            // find the shortest bank prefix [0, t_cut] holding at least trig_capacity triggers from the
            // per-template counts and filter that prefix again into a buffer that takes all of its triggers.
            std::vector<unsigned int> cnt((size_t)nt);
            CU(cudaMemcpyAsync(cnt.data(), c->d_tcount, sizeof(unsigned int) * (size_t)nt, cudaMemcpyDeviceToHost, c->stream));
            CU(cudaStreamSynchronize(c->stream));
            int64_t cum = 0, t_cut = 0;
            for (; t_cut < nt; ++t_cut) { cum += cnt[(size_t)t_cut]; if (cum >= trig_capacity) break; }
            int64_t need = 1;
            while (need < cum) need <<= 1;
            if ((rc = grow(c, c->d_trig, c->trig_cap, need))) return rc;
            CU(cudaMemsetAsync(c->d_cursor, 0, sizeof(unsigned long long), c->stream));
            CU(cudaMemsetAsync(c->d_tcount, 0, sizeof(unsigned int) * (size_t)nt, c->stream));
            const int prof = c->profiling;
            c->profiling = 0;                           // the repeat is not part of the per-pass timing
            rc = run_bank_passes(c, t_cut + 1, c->trig_cap, w, j_min);
            c->profiling = prof;
            if (rc) return rc;
            on_device = cum;
        }
        if ((rc = sort_triggers(c, on_device))) return rc;
        CU(cudaMemcpyAsync(trig_out, c->d_trig, sizeof(TrigOut) * (size_t)kept, out_kind, c->stream));
    }
    CU(cudaMemcpyAsync(peaks_out, c->d_peaks, sizeof(PeakOut) * (size_t)nt, out_kind, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return (found > trig_capacity) ? CBMF_WTRUNC : CBMF_OK;
}

// One bank pass over the segment whose weights are w (default: the context's), samples j < j_min excluded: filter,
// count, sort and deliver.  Outputs go to host or device pointers (out_kind); *found_out = all triggers found.
static int bank_filter(cbmf_ctx* c, int64_t nt, const c2* w, int j_min, void* peaks_out, void* trig_out,
                       int64_t trig_capacity, int64_t* found_out, cudaMemcpyKind out_kind)
{
    int rc;
    // device trigger buffer: capacity rounded up to a power of two (bitonic padding), >= 1
    int64_t tcap = 1;
    while (tcap < trig_capacity) tcap <<= 1;
    if ((rc = grow(c, c->d_trig, c->trig_cap, tcap))) return rc;
    CU(cudaMemsetAsync(c->d_cursor, 0, sizeof(unsigned long long), c->stream));
    CU(cudaMemsetAsync(c->d_tcount, 0, sizeof(unsigned int) * (size_t)nt, c->stream));
    c->ev_used[0] = c->ev_used[1] = 0;
    if ((rc = run_bank_passes(c, nt, c->trig_cap, w, j_min))) return rc;

    // trigger count back to the host, then sort what was kept
    unsigned long long found_u = 0;
    CU(cudaMemcpyAsync(&found_u, c->d_cursor, sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if ((rc = ev_collect(c))) return rc;
    const int64_t found = (int64_t)found_u;
    if (found_out) *found_out = found;
    return collect_triggers(c, nt, w, j_min, found, peaks_out, trig_out, trig_capacity, out_kind);
}

// The plain bank call.  Everything is enqueued behind one another -- status reset, template setup, the launch pairs
// (which return at once if the setup found an invalid template), a single-block sort of up to TRIG_SMALL triggers with
// the count read on the device, the result copies -- and the host waits ONCE; only a bank with more triggers than
// that, or than the list holds, goes through the general collection (bank_filter's tail) afterwards.
static int filter_bank_impl(cbmf_ctx* c, const double* bank_dev, int64_t nt, float thr,
                            void* peaks_out, void* trig_out, int64_t trig_capacity,
                            int64_t* n_trig_found, cudaMemcpyKind out_kind)
{
    if (n_trig_found) *n_trig_found = 0;
    c->last_bad = -1;
    if (nt == 0) return CBMF_OK;
    int rc;
    if ((rc = grow(c, c->d_coef, c->coef_cap, nt))) return rc;
    if ((rc = grow(c, c->d_peaks, c->peaks_cap, nt))) return rc;
    if ((rc = grow(c, c->d_tcount, c->tcount_cap, nt))) return rc;
    int64_t tcap = 1;
    while (tcap < trig_capacity) tcap <<= 1;
    if ((rc = grow(c, c->d_trig, c->trig_cap, tcap))) return rc;
    const bool to_host = (out_kind == cudaMemcpyDeviceToHost);
    const int64_t n_fast = trig_capacity < TRIG_SMALL ? trig_capacity : TRIG_SMALL;      // triggers the fast path delivers
    const size_t b_status = 32, b_peaks = sizeof(PeakOut) * (size_t)nt, b_trig = sizeof(TrigOut) * (size_t)n_fast;
    if (b_status + b_peaks + b_trig > c->stage_bytes) {
        if (c->h_stage) { CU(cudaFreeHost(c->h_stage)); c->h_stage = nullptr; c->stage_bytes = 0; }
        CU(cudaMallocHost(&c->h_stage, b_status + b_peaks + b_trig));
        c->stage_bytes = b_status + b_peaks + b_trig;
    }
    unsigned long long* h_status = reinterpret_cast<unsigned long long*>(c->h_stage);
    unsigned char* h_peaks = c->h_stage + b_status;
    unsigned char* h_trig = h_peaks + b_peaks;

    h_status[0] = 0ULL; h_status[1] = (unsigned long long)NO_BAD_TEMPLATE;
    CU(cudaMemcpyAsync(c->d_cursor, h_status, 16, cudaMemcpyHostToDevice, c->stream));            // cursor = 0, bad = none
    SetupArgs sa;
    sa.bank = bank_dev; sa.prefix = c->d_prefix; sa.coef = c->d_coef; sa.n_templates = (int)nt;
    sa.n_half = (int)(c->n / 2); sa.k_lo = c->k_lo; sa.n_over_fs = (double)c->n / c->fs; sa.df = c->df;
    sa.threshold = thr; sa.err_flag = c->d_err; sa.bad_idx = c->d_bad; sa.tcount = c->d_tcount; sa.pn_half_order = c->pn_half_order;
    template_setup_kernel<<<(unsigned)((nt + 127) / 128), 128, 0, c->stream>>>(sa);
    CU(cudaGetLastError());
    c->launches += 1;
    c->ev_used[0] = c->ev_used[1] = 0;
    if ((rc = run_bank_passes(c, nt, c->trig_cap))) return rc;
    const int sort_limit = (int)(c->trig_cap < TRIG_SMALL ? c->trig_cap : TRIG_SMALL);
    CU(ensure_smem_attr(c, trig_sort_small_dev_kernel, trig_sort_dev_smem()));
    trig_sort_small_dev_kernel<<<1, 1024, trig_sort_dev_smem(), c->stream>>>(c->d_trig, c->d_cursor, c->d_bad, sort_limit,
                                                                              c->d_tcount, (int)nt);
    CU(cudaGetLastError());
    c->launches += 1;
    CU(cudaMemcpyAsync(h_status, c->d_cursor, b_status, cudaMemcpyDeviceToHost, c->stream));
    if (to_host) {
        CU(cudaMemcpyAsync(h_peaks, c->d_peaks, b_peaks, cudaMemcpyDeviceToHost, c->stream));
        if (b_trig && trig_out) CU(cudaMemcpyAsync(h_trig, c->d_trig, b_trig, cudaMemcpyDeviceToHost, c->stream));
    }
    CU(cudaStreamSynchronize(c->stream));
    if ((rc = ev_collect(c))) return rc;
    {   // input checks that cbmf_set_psd_dev / cbmf_load_segment_dev left pending come back with the same copy
        const int* errs = reinterpret_cast<const int*>(h_status + 2);
        const bool bad_psd = c->pend_psd && errs[0], bad_seg = c->pend_seg && errs[1];
        c->pend_psd = c->pend_seg = false;
        if (bad_psd) { c->have_psd = false; c->have_seg = false; return CBMF_EINVAL; }
        if (bad_seg) { c->have_seg = false; return CBMF_EINVAL; }
    }
    if ((long long)h_status[1] != NO_BAD_TEMPLATE) { c->last_bad = (int64_t)h_status[1]; return CBMF_EINVAL; }
    const int64_t found = (int64_t)h_status[0];
    if (n_trig_found) *n_trig_found = found;
    const int64_t kept = found < trig_capacity ? found : trig_capacity;
    if (found <= sort_limit && found <= trig_capacity) {
        // the common case: the sorted list is complete
        if (to_host) {
            memcpy(peaks_out, h_peaks, b_peaks);
            if (kept > 0 && trig_out) memcpy(trig_out, h_trig, sizeof(TrigOut) * (size_t)kept);
        } else {
            if (kept > 0 && trig_out) CU(cudaMemcpyAsync(trig_out, c->d_trig, sizeof(TrigOut) * (size_t)kept, out_kind, c->stream));
            CU(cudaMemcpyAsync(peaks_out, c->d_peaks, b_peaks, out_kind, c->stream));
            CU(cudaStreamSynchronize(c->stream));
        }
        return CBMF_OK;
    }
    // many triggers: the general collection (sort of any size, truncated lists)
    return collect_triggers(c, nt, nullptr, 0, found, peaks_out, trig_out, trig_capacity, out_kind);
}

static int filter_args_ok(cbmf_ctx* c, const void* bank, int64_t nt, float thr, void* peaks,
                          void* trig, int64_t cap)
{
    if (!c || nt < 0 || cap < 0) return CBMF_EINVAL;
    if (nt > 0 && (!bank || !peaks)) return CBMF_EINVAL;
    if (cap > 0 && !trig) return CBMF_EINVAL;
    if (!(thr >= 0.f)) return CBMF_EINVAL;                 // negative or NaN
    if (nt > 0x7FFFFFFF) return CBMF_EINVAL;
    if (!c->have_psd || !c->have_seg) return CBMF_ESTATE;
    return CBMF_OK;
}

extern "C" int cbmf_filter_bank_dev(cbmf_ctx* c, const cbmf_template* bank_dev, int64_t nt, float thr,
                                    cbmf_peak* peaks_out_dev, cbmf_trigger* trig_out_dev,
                                    int64_t trig_capacity, int64_t* n_trig_found)
{
    int rc = filter_args_ok(c, bank_dev, nt, thr, peaks_out_dev, trig_out_dev, trig_capacity);
    if (rc) return rc;
    DeviceGuard g(c->device);
    return filter_bank_impl(c, (const double*)bank_dev, nt, thr, peaks_out_dev, trig_out_dev,
                            trig_capacity, n_trig_found, cudaMemcpyDeviceToDevice);
}

extern "C" int cbmf_filter_bank(cbmf_ctx* c, const cbmf_template* bank, int64_t nt, float thr,
                                cbmf_peak* peaks_out, cbmf_trigger* trig_out, int64_t trig_capacity,
                                int64_t* n_trig_found)
{
    int rc = filter_args_ok(c, bank, nt, thr, peaks_out, trig_out, trig_capacity);
    if (rc) return rc;
    if (n_trig_found) *n_trig_found = 0;
    if (nt == 0) return CBMF_OK;
    DeviceGuard g(c->device);
    if ((rc = grow(c, c->d_bank, c->bank_cap, 2 * nt))) return rc;
    CU(cudaMemcpyAsync(c->d_bank, bank, sizeof(cbmf_template) * (size_t)nt, cudaMemcpyHostToDevice, c->stream));
    return filter_bank_impl(c, c->d_bank, nt, thr, peaks_out, trig_out, trig_capacity, n_trig_found,
                            cudaMemcpyDeviceToHost);
}

// ======================================================================= NEXT-1: clustered bank call
// The bank loop of cbmf_filter_bank with the host-side reduction of PAPER.md:103 / :131 behind it: every launch pair
// (sub-batch) writes its raw triggers to its own device region; a copy to pinned host memory follows the pair on its
// stream; the host enqueues pairs up to PIPE_RING ahead and, pair by pair as their copies complete, sorts and
// clusters the triggers (cluster.h) WHILE the GPU filters the following pairs.
namespace {
constexpr int PIPE_RING = 32;                 // pairs enqueued ahead of the one the host is clustering
constexpr int PAIR_TRIG_CAP = 4096;           // raw triggers kept per launch pair (64 KiB per copy)

int pipe_alloc(cbmf_ctx* c)
{
    if (c->d_ptrig) return CBMF_OK;
    CU(cudaMalloc(&c->d_ptrig, sizeof(TrigOut) * (size_t)CBMF_MAX_STREAMS * PAIR_TRIG_CAP));
    CU(cudaMalloc(&c->d_pcursor, sizeof(unsigned long long) * CBMF_MAX_STREAMS));
    CU(cudaMallocHost(&c->h_ptrig, sizeof(TrigOut) * (size_t)PIPE_RING * PAIR_TRIG_CAP));
    CU(cudaMallocHost(&c->h_pcursor, sizeof(unsigned long long) * PIPE_RING));
    for (int i = 0; i < PIPE_RING; ++i) CU(cudaEventCreateWithFlags(&c->ev_pipe[i], cudaEventDisableTiming));
    return CBMF_OK;
}
}  // namespace

extern "C" int cbmf_cluster_triggers(const cbmf_trigger* trig, int64_t n_trig, int64_t n_samples, int64_t window_samples,
                                     cbmf_trigger* events_out, int64_t event_capacity, int64_t* n_events)
{
    if ((!trig && n_trig) || n_trig < 0 || n_samples <= 0 || window_samples < 0 || event_capacity < 0 || !n_events)
        return CBMF_EINVAL;
    if (event_capacity > 0 && !events_out) return CBMF_EINVAL;
    *n_events = 0;
    std::vector<HostTrig> ev;
    if (!cluster_sorted(reinterpret_cast<const HostTrig*>(trig), n_trig, n_samples, window_samples, ev)) return CBMF_EINVAL;
    const int64_t n = (int64_t)ev.size(), kept = n < event_capacity ? n : event_capacity;
    if (kept) memcpy(events_out, ev.data(), sizeof(HostTrig) * (size_t)kept);
    *n_events = n;
    return n > event_capacity ? CBMF_WTRUNC : CBMF_OK;
}

extern "C" int cbmf_filter_bank_clustered(cbmf_ctx* c, const cbmf_template* bank, int64_t nt, float thr,
                                          int64_t window_samples, cbmf_peak* peaks_out, cbmf_trigger* events_out,
                                          int64_t event_capacity, int64_t* n_events, int64_t* n_trig_found)
{
    int rc = filter_args_ok(c, bank, nt, thr, peaks_out, events_out, event_capacity);
    if (rc) return rc;
    if (window_samples < 0 || !n_events) return CBMF_EINVAL;
    *n_events = 0;
    if (n_trig_found) *n_trig_found = 0;
    c->last_bad = -1;
    if (nt == 0) return CBMF_OK;
    DeviceGuard g(c->device);
    if ((rc = check_pending(c))) return rc;
    if ((rc = grow(c, c->d_bank, c->bank_cap, 2 * nt))) return rc;
    if ((rc = pipe_alloc(c))) return rc;
    CU(cudaMemcpyAsync(c->d_bank, bank, sizeof(cbmf_template) * (size_t)nt, cudaMemcpyHostToDevice, c->stream));
    if ((rc = bank_setup(c, c->d_bank, nt, thr))) return rc;
    CU(cudaMemsetAsync(c->d_tcount, 0, sizeof(unsigned int) * (size_t)nt, c->stream));

    const int sb = eff_sub_batch(c, nt), ns = c->n_streams;
    const size_t ncand = cand_per_template(c);
    const int64_t n_pairs = (nt + sb - 1) / sb;
    // this call records no per-pass events: cbmf_last_pass_time / cbmf_debug_timeline read empty after it
    auto reset_profile = [&]() {
        for (int w = 0; w < 2; ++w) { c->ev_used[w] = 0; c->last_ms[w] = 0; c->last_launches[w] = 0; c->timeline[w].clear(); }
    };
    reset_profile();
    CU(cudaEventRecord(c->ev_fork, c->stream));
    for (int s = 0; s < ns; ++s) CU(cudaStreamWaitEvent(c->aux[s], c->ev_fork, 0));

    std::vector<HostTrig> events;
    std::vector<int64_t> overflow;              // pairs whose raw list did not fit PAIR_TRIG_CAP: filtered again below
    int64_t found_total = 0;
    auto enqueue = [&](int64_t pair) -> int {
        const int64_t t0 = pair * sb;
        const int nb = (int)((nt - t0 < sb) ? (nt - t0) : sb);
        const int slot = (int)(pair % ns), ring = (int)(pair % PIPE_RING);
        cudaStream_t st = c->aux[slot];
        c2* Y = c->d_Y + (size_t)slot * c->max_sub_batch * (size_t)c->n;
        CU(cudaMemsetAsync(c->d_pcursor + slot, 0, sizeof(unsigned long long), st));
        P1Args a1; memset(&a1, 0, sizeof(a1));
        a1.w = c->d_w; a1.u = c->d_u; a1.lnk = c->d_lnk; a1.coef = c->d_coef + t0; a1.Y = Y; a1.err_flag = c->d_err; a1.use_series = c->k_lo;
        CU(launch_p1<LOAD_GEN>(c, st, a1, nb));
        P2Args a2; memset(&a2, 0, sizeof(a2));
        a2.Y = Y; a2.coef = c->d_coef + t0;
        a2.cand = c->d_cand + (size_t)slot * c->max_sub_batch * ncand;
        a2.best_key = c->d_key + (size_t)slot * c->max_sub_batch;
        a2.done_ctr = c->d_done + (size_t)slot * c->max_sub_batch; a2.peaks = c->d_peaks + t0;
        a2.trig = c->d_ptrig + (size_t)slot * PAIR_TRIG_CAP;
        a2.trig_cursor = c->d_pcursor + slot; a2.trig_cap = PAIR_TRIG_CAP;
        a2.trig_count = c->d_tcount + t0;
        a2.tmpl_base = (int)t0;
        CU(launch_p2<EPI_MAX>(c, st, a2, nb));
        c->launches += 2;
        CU(cudaMemcpyAsync(c->h_pcursor + ring, c->d_pcursor + slot, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
        CU(cudaMemcpyAsync(c->h_ptrig + (size_t)ring * PAIR_TRIG_CAP, a2.trig, sizeof(TrigOut) * PAIR_TRIG_CAP,
                           cudaMemcpyDeviceToHost, st));
        CU(cudaEventRecord(c->ev_pipe[ring], st));
        return CBMF_OK;
    };
    auto key_less = [](const HostTrig& a, const HostTrig& b) {
        return a.template_idx != b.template_idx ? a.template_idx < b.template_idx : a.sample_idx < b.sample_idx;
    };
    auto pipeline = [&]() -> int {
        int64_t next_enq = 0;
        for (int64_t done = 0; done < n_pairs; ++done) {
            // ns pairs share the ring slot's stream order; keep the ring one short of full so a slot is never re-armed
            // before the host has consumed it
            while (next_enq < n_pairs && next_enq - done < PIPE_RING - 1)
                if (int e = enqueue(next_enq++)) return e;
            const int ring = (int)(done % PIPE_RING);
            CU(cudaEventSynchronize(c->ev_pipe[ring]));
            const int64_t found = (int64_t)c->h_pcursor[ring];
            found_total += found;
            if (found > PAIR_TRIG_CAP) { overflow.push_back(done); continue; }
            HostTrig* t = reinterpret_cast<HostTrig*>(c->h_ptrig + (size_t)ring * PAIR_TRIG_CAP);
            std::sort(t, t + found, key_less);
            if (!cluster_sorted(t, found, c->n, window_samples, events)) return CBMF_ECUDA;  // cannot happen: device indices are in range
        }
        return CBMF_OK;
    };
    rc = pipeline();
    if (rc) {
        // leave nothing running on the internal streams: a later call reuses d_Y, d_w and the pair regions
        for (int s = 0; s < ns; ++s) cudaStreamSynchronize(c->aux[s]);
        cudaStreamSynchronize(c->stream);
        cudaGetLastError();
        return rc;
    }
    for (int s = 0; s < ns; ++s) {
        CU(cudaEventRecord(c->ev_join[s], c->aux[s]));
        CU(cudaStreamWaitEvent(c->stream, c->ev_join[s], 0));
    }
    CU(cudaMemcpyAsync(peaks_out, c->d_peaks, sizeof(PeakOut) * (size_t)nt, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (!overflow.empty()) {
        // A pair with more raw triggers than its region holds (a loud transient): its templates are filtered again
        // through the plain call, in runs of consecutive templates whose trigger counts (known from the first pass)
        // add up to at most RERUN_TRIG, each run with a list that takes all of its triggers, and clustered.
        constexpr int64_t RERUN_TRIG = int64_t(1) << 22;          // 64 MiB of trigger list per re-run
        std::vector<unsigned int> cnt((size_t)nt);
        CU(cudaMemcpyAsync(cnt.data(), c->d_tcount, sizeof(unsigned int) * (size_t)nt, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));                      // the re-runs below reuse d_tcount
        std::vector<PeakOut> pk;
        std::vector<HostTrig> raw;
        for (int64_t pair : overflow) {
            const int64_t t0 = pair * sb, t_end = (nt - t0 < sb) ? nt : t0 + sb;
            for (int64_t a = t0; a < t_end;) {
                int64_t b = a, sum = 0;
                do { sum += cnt[(size_t)b]; ++b; } while (b < t_end && sum + (int64_t)cnt[(size_t)b] <= RERUN_TRIG);
                if (sum > 0) {
                    pk.resize((size_t)(b - a));
                    raw.resize((size_t)sum);
                    int64_t nf = 0;
                    rc = filter_bank_impl(c, c->d_bank + 2 * a, b - a, thr, pk.data(), raw.data(), sum, &nf, cudaMemcpyDeviceToHost);
                    if (rc < 0) return rc;
                    const int64_t got = nf < sum ? nf : sum;       // the same kernels on the same input: nf == sum
                    for (int64_t j = 0; j < got; ++j) raw[(size_t)j].template_idx += (int32_t)a;
                    if (!cluster_sorted(raw.data(), got, c->n, window_samples, events)) return CBMF_ECUDA;
                }
                a = b;
            }
        }
        std::stable_sort(events.begin(), events.end(), key_less);
        reset_profile();                                           // the re-runs are not the call's passes
    }
    const int64_t n_ev = (int64_t)events.size(), kept = n_ev < event_capacity ? n_ev : event_capacity;
    if (kept) memcpy(events_out, events.data(), sizeof(HostTrig) * (size_t)kept);
    *n_events = n_ev;
    if (n_trig_found) *n_trig_found = found_total;
    return n_ev > event_capacity ? CBMF_WTRUNC : CBMF_OK;
}

// ======================================================================= NEXT-2: segment streaming
extern "C" int cbmf_filter_stream(cbmf_ctx* c, const float* samples, int64_t n_total, const cbmf_template* bank,
                                  int64_t nt, float thr, int64_t discard, cbmf_peak* peaks_out,
                                  cbmf_trigger* trig_out, int64_t trig_capacity, int64_t* seg_offsets_out,
                                  int64_t* n_trig_found, int64_t* n_segments)
{
    if (!c || !samples || !n_segments || nt < 0 || trig_capacity < 0) return CBMF_EINVAL;
    if (nt > 0 && (!bank || !peaks_out)) return CBMF_EINVAL;
    if (trig_capacity > 0 && !trig_out) return CBMF_EINVAL;
    if (!(thr >= 0.f) || nt > 0x7FFFFFFF) return CBMF_EINVAL;
    if (discard < 0 || discard >= c->n || n_total < c->n) return CBMF_EINVAL;
    if (!c->have_psd) return CBMF_ESTATE;
    const int64_t n = c->n, hop = n - discard, n_seg = (n_total - n) / hop + 1;
    *n_segments = n_seg;
    if (n_trig_found) *n_trig_found = 0;
    if (seg_offsets_out) seg_offsets_out[0] = 0;
    c->last_bad = -1;
    DeviceGuard g(c->device);
    int rc;
    if ((rc = check_pending(c))) return rc;
    c->have_seg = false;                       // the context's own segment slot is used as buffer 0 of the stream
    if (!c->d_w2) {
        CU(cudaMalloc(&c->d_w2, sizeof(c2) * (size_t)(n / 2)));
        CU(cudaMalloc(&c->d_segY, sizeof(c2) * (size_t)n));
        CU(cudaMalloc(&c->d_segin, sizeof(float) * (size_t)n));
        CU(cudaMalloc(&c->d_segerr, sizeof(int)));
        CU(cudaStreamCreateWithFlags(&c->seg_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) CU(cudaEventCreateWithFlags(&c->ev_seg_ready[i], cudaEventDisableTiming));
    }
    if (nt > 0) {
        if ((rc = grow(c, c->d_bank, c->bank_cap, 2 * nt))) return rc;
        CU(cudaMemcpyAsync(c->d_bank, bank, sizeof(cbmf_template) * (size_t)nt, cudaMemcpyHostToDevice, c->stream));
        if ((rc = bank_setup(c, c->d_bank, nt, thr))) return rc;     // the constants serve every segment
    }
    c2* wbuf[2] = {c->d_w, c->d_w2};
    auto load = [&](int64_t s) -> int {       // segment s: host -> device -> w[s % 2], all on the loader stream
        CU(cudaMemcpyAsync(c->d_segin, samples + s * hop, sizeof(float) * (size_t)n, cudaMemcpyHostToDevice, c->seg_stream));
        int r = enqueue_load_segment(c, c->d_segin, wbuf[s & 1], c->d_segY, c->seg_stream, c->d_segerr);
        if (r) return r;
        CU(cudaEventRecord(c->ev_seg_ready[s & 1], c->seg_stream));
        return CBMF_OK;
    };
    CU(cudaStreamSynchronize(c->stream));
    if ((rc = load(0))) return rc;
    int64_t written = 0, found_total = 0;
    bool truncated = false;
    for (int64_t s = 0; s < n_seg; ++s) {
        // the loader has had the previous bank's time to finish: its error flag first (a NaN / Inf sample)
        int err = 0;
        CU(cudaMemcpyAsync(&err, c->d_segerr, sizeof(int), cudaMemcpyDeviceToHost, c->seg_stream));
        CU(cudaStreamSynchronize(c->seg_stream));
        if (err) return CBMF_EINVAL;
        // Segment s + 1 is loaded and transformed on the loader stream WHILE the bank runs on segment s
        // (keep the data on the device; the other buffer was last read by the bank of segment s - 1,
        // which has been collected).  The bank of segment s is enqueued first so that it owns the SMs.
        if (nt == 0) { if (s + 1 < n_seg && (rc = load(s + 1))) return rc; if (seg_offsets_out) seg_offsets_out[s + 1] = 0; continue; }
        const int64_t room = trig_capacity - written;
        int64_t found = 0;
        CU(cudaStreamWaitEvent(c->stream, c->ev_seg_ready[s & 1], 0));      // the bank forks from the context's stream
        // bank_filter enqueues the whole bank and then waits for it; the next load must be enqueued in between, so
        // hand it over as a hook that run_bank_passes calls after its last launch
        c->after_enqueue = (s + 1 < n_seg) ? 1 : 0;
        c->after_enqueue_seg = s + 1;
        struct Hook { decltype(load)* f; } hk{&load};
        c->after_enqueue_fn = [](void* p, int64_t seg) -> int { return (*static_cast<Hook*>(p)->f)(seg); };
        c->after_enqueue_arg = &hk;
        rc = bank_filter(c, nt, wbuf[s & 1], (int)discard, peaks_out + s * nt, trig_out ? trig_out + written : nullptr,
                         room > 0 ? room : 0, &found, cudaMemcpyDeviceToHost);
        c->after_enqueue = 0;
        c->after_enqueue_fn = nullptr;
        if (rc < 0) return rc;
        if (rc == CBMF_WTRUNC) truncated = true;
        found_total += found;
        written += (found < room) ? found : (room > 0 ? room : 0);
        if (seg_offsets_out) seg_offsets_out[s + 1] = written;
    }
    CU(cudaStreamSynchronize(c->seg_stream));
    if (n_trig_found) *n_trig_found = found_total;
    return truncated ? CBMF_WTRUNC : CBMF_OK;
}

// ======================================================================= NEXT-4: chi-squared veto
extern "C" int cbmf_chisq(cbmf_ctx* c, const cbmf_template* bank, int64_t nt, const int32_t* sample_idx, int p_bands,
                          float* chisq_out, double* zl_out)
{
    if (!c || nt < 0 || (nt > 0 && (!bank || !sample_idx || !chisq_out))) return CBMF_EINVAL;
    if (p_bands < 1 || p_bands > CHISQ_MAX_BANDS || nt > 65535) return CBMF_EINVAL;
    if (!c->have_psd || !c->have_seg) return CBMF_ESTATE;
    for (int64_t i = 0; i < nt; ++i) if (sample_idx[i] >= c->n) return CBMF_EINVAL;       // < 0: no sample, chi^2 = 0
    if (nt == 0) return CBMF_OK;
    DeviceGuard g(c->device);
    int rc;
    if ((rc = check_pending(c))) return rc;
    if ((rc = grow(c, c->d_bank, c->bank_cap, 2 * nt))) return rc;
    CU(cudaMemcpyAsync(c->d_bank, bank, sizeof(cbmf_template) * (size_t)nt, cudaMemcpyHostToDevice, c->stream));
    if ((rc = bank_setup(c, c->d_bank, nt, 0.f))) return rc;
    const int p = p_bands;
    const size_t b_edges = sizeof(int) * (size_t)nt * (p + 1), b_idx = sizeof(int) * (size_t)nt;
    const size_t b_zl = sizeof(double) * 2 * (size_t)nt * p, b_chi = sizeof(float) * (size_t)nt;
    if ((rc = grow_scratch(c, b_zl + b_edges + b_idx + b_chi + 64))) return rc;
    double* d_zl = (double*)c->d_scratch;
    int* d_edges = (int*)(d_zl + 2 * (size_t)nt * p);
    int* d_idx = d_edges + (size_t)nt * (p + 1);
    float* d_chi = (float*)(d_idx + nt);
    CU(cudaMemcpyAsync(d_idx, sample_idx, b_idx, cudaMemcpyHostToDevice, c->stream));
    const int ne = (int)nt * (p + 1);
    chisq_edges_kernel<<<(ne + 127) / 128, 128, 0, c->stream>>>(c->d_coef, c->d_prefix, p, d_edges, (int)nt);
    CU(cudaGetLastError());
    chisq_bands_kernel<<<dim3((unsigned)p, (unsigned)nt), 256, 0, c->stream>>>(c->d_w, c->d_u, c->d_lnk, c->d_coef, d_edges, d_idx, p,
                                                                                 c->log2n, d_zl);
    CU(cudaGetLastError());
    chisq_finish_kernel<<<(unsigned)((nt + 127) / 128), 128, 0, c->stream>>>(c->d_coef, c->d_prefix, d_edges, d_zl, p, d_chi, (int)nt);
    CU(cudaGetLastError());
    c->launches += 3;
    CU(cudaMemcpyAsync(chisq_out, d_chi, b_chi, cudaMemcpyDeviceToHost, c->stream));
    if (zl_out) CU(cudaMemcpyAsync(zl_out, d_zl, b_zl, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return CBMF_OK;
}

// ======================================================================= NEXT-3, second part: time-domain templates
// The paper's own template path (td.cuh): per step of up to TD_STEP templates
//   generate -> forward FFT (one complex transform for both polarisations) -> normalisation sums -> two-sided product
//   -> inverse FFT -> the arg-max / threshold epilogue of the SPA path on rho^2 = |c_+/sigma_+ + i c_x/sigma_x|^2,
// everything on the context's stream.  It is the comparison path, not the tuned one: ~100 bytes of HBM traffic per
// sample and template against 16 for the SPA path.
namespace {
constexpr int TD_STEP = 16;

int td_alloc(cbmf_ctx* c, int64_t nt, int step)
{
    int rc;
    if ((rc = grow(c, c->d_td, c->td_cap, nt))) return rc;
    if ((rc = grow(c, c->d_tdnorm, c->tdnorm_cap, 2 * nt))) return rc;
    if ((rc = grow(c, c->d_tdinv, c->tdinv_cap, nt))) return rc;
    if ((rc = grow(c, c->d_tdU, c->tdU_cap, (int64_t)step * c->n))) return rc;
    const size_t nh = (size_t)c->n / 2;
    if (!c->d_winv) CU(cudaMalloc(&c->d_winv, sizeof(float) * nh));
    if (!c->d_wd) CU(cudaMalloc(&c->d_wd, sizeof(c2) * nh));
    return CBMF_OK;
}

int td_setup(cbmf_ctx* c, const double* bank_dev, int64_t nt, float thr)
{
    TdSetupArgs sa;
    sa.bank = bank_dev; sa.td = c->d_td; sa.coef = c->d_coef; sa.norm = c->d_tdnorm; sa.tcount = c->d_tcount;
    sa.n_templates = (int)nt; sa.n_half = (int)(c->n / 2); sa.k_lo = c->k_lo; sa.pn_half_order = c->pn_half_order;
    sa.f_low = c->f_low; sa.seg_seconds = (double)c->n * c->dt; sa.threshold = thr;
    sa.err_flag = c->d_err; sa.bad_idx = c->d_bad;
    td_setup_kernel<<<(unsigned)((nt + 63) / 64), 64, 0, c->stream>>>(sa);
    CU(cudaGetLastError());
    c->launches += 1;
    return CBMF_OK;
}

// One pass over the bank into c->d_peaks / c->d_trig (dev_cap entries); the total count stays in c->d_cursor.
int td_run(cbmf_ctx* c, int64_t nt, int step, int64_t dev_cap)
{
    const int n = (int)c->n, nh = n / 2;
    const size_t ncand = cand_per_template(c);
    int gx = (nh + 255) / 256; if (gx > 1184) gx = 1184;
    for (int64_t t0 = 0; t0 < nt; t0 += step) {
        const int nb = (int)((nt - t0 < step) ? (nt - t0) : step);
        td_generate_kernel<<<dim3((unsigned)((n + 255) / 256), (unsigned)nb), 256, 0, c->stream>>>(c->d_td + t0, c->d_tdU, n, c->dt, -1.0f);
        CU(cudaGetLastError());
        P1Args a1; memset(&a1, 0, sizeof(a1));
        a1.in_c = c->d_tdU; a1.Y = c->d_Y; a1.err_flag = c->d_err;
        CU(launch_p1<LOAD_CPLX>(c, c->stream, a1, nb));
        P2Args a2; memset(&a2, 0, sizeof(a2));
        a2.Y = c->d_Y; a2.z_out = c->d_tdU;
        CU(launch_p2<EPI_STORE>(c, c->stream, a2, nb));
        td_norm_kernel<<<dim3(64, (unsigned)nb), 256, 0, c->stream>>>(c->d_tdU, c->d_winv, c->d_tdnorm + 2 * t0, n, c->k_lo, (float)c->dt);
        CU(cudaGetLastError());
        td_norm_finish_kernel<<<1, 64, 0, c->stream>>>(c->d_tdnorm + 2 * t0, c->d_coef + t0, c->d_tdinv + t0, nb);
        CU(cudaGetLastError());
        td_product_kernel<<<dim3((unsigned)gx, (unsigned)nb), 256, 0, c->stream>>>(c->d_tdU, c->d_wd, c->d_tdinv + t0, n, c->k_lo, (float)c->dt);
        CU(cudaGetLastError());
        CU(launch_p1<LOAD_CPLX>(c, c->stream, a1, nb));
        P2Args a3; memset(&a3, 0, sizeof(a3));
        a3.Y = c->d_Y; a3.coef = c->d_coef + t0; a3.cand = c->d_cand; a3.best_key = c->d_key; a3.done_ctr = c->d_done;
        a3.peaks = c->d_peaks + t0; a3.trig = c->d_trig; a3.trig_cursor = c->d_cursor; a3.trig_cap = (unsigned long long)dev_cap;
        a3.trig_count = c->d_tcount + t0; a3.tmpl_base = (int)t0; a3.j_min = 0; a3.bad = c->d_bad;
        (void)ncand;
        CU(launch_p2<EPI_MAX>(c, c->stream, a3, nb));
        c->launches += 8;
    }
    return CBMF_OK;
}
}  // namespace

extern "C" int cbmf_filter_bank_td(cbmf_ctx* c, const cbmf_template* bank, int64_t nt, float thr,
                                   cbmf_peak* peaks_out, cbmf_trigger* trig_out, int64_t trig_capacity,
                                   int64_t* n_trig_found)
{
    int rc = filter_args_ok(c, bank, nt, thr, peaks_out, trig_out, trig_capacity);
    if (rc) return rc;
    if (n_trig_found) *n_trig_found = 0;
    c->last_bad = -1;
    if (nt == 0) return CBMF_OK;
    DeviceGuard g(c->device);
    if ((rc = check_pending(c))) return rc;
    const int step = c->sub_batch < TD_STEP ? c->sub_batch : TD_STEP;
    if ((rc = grow(c, c->d_bank, c->bank_cap, 2 * nt))) return rc;
    if ((rc = grow(c, c->d_coef, c->coef_cap, nt))) return rc;
    if ((rc = grow(c, c->d_peaks, c->peaks_cap, nt))) return rc;
    if ((rc = grow(c, c->d_tcount, c->tcount_cap, nt))) return rc;
    if ((rc = td_alloc(c, nt, step))) return rc;
    int64_t tcap = 1;
    while (tcap < trig_capacity) tcap <<= 1;
    if ((rc = grow(c, c->d_trig, c->trig_cap, tcap))) return rc;
    CU(cudaMemcpyAsync(c->d_bank, bank, sizeof(cbmf_template) * (size_t)nt, cudaMemcpyHostToDevice, c->stream));
    const int nh = (int)(c->n / 2);
    td_tables_kernel<<<(unsigned)((nh + 255) / 256), 256, 0, c->stream>>>(c->d_wfac, c->d_w, c->d_winv, c->d_wd, nh, c->k_lo, c->df, c->dt);
    CU(cudaGetLastError());
    c->launches += 1;
    int64_t found = 0;
    for (int attempt = 0; attempt < 2; ++attempt) {
        unsigned long long status[2] = {0ULL, (unsigned long long)NO_BAD_TEMPLATE};
        CU(cudaMemcpyAsync(c->d_cursor, status, sizeof(status), cudaMemcpyHostToDevice, c->stream));
        CU(cudaMemsetAsync(c->d_err, 0, sizeof(int), c->stream));
        if ((rc = td_setup(c, c->d_bank, nt, thr))) return rc;
        CU(cudaMemcpyAsync(status, c->d_cursor, sizeof(status), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        if ((long long)status[1] != NO_BAD_TEMPLATE) { c->last_bad = (int64_t)status[1]; return CBMF_EINVAL; }
        if ((rc = td_run(c, nt, step, c->trig_cap))) return rc;
        CU(cudaMemcpyAsync(status, c->d_cursor, sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        found = (int64_t)status[0];
        if (found <= c->trig_cap || !trig_out || trig_capacity == 0) break;
        // the device list is incomplete: once more with room for all of them (the kept ones are the FIRST in order)
        int64_t need = 1;
        while (need < found) need <<= 1;
        if ((rc = grow(c, c->d_trig, c->trig_cap, need))) return rc;
    }
    if (n_trig_found) *n_trig_found = found;
    const int64_t kept = found < trig_capacity ? found : trig_capacity;
    if (kept > 0 && trig_out) {
        if ((rc = sort_triggers(c, found))) return rc;
        CU(cudaMemcpyAsync(trig_out, c->d_trig, sizeof(TrigOut) * (size_t)kept, cudaMemcpyDeviceToHost, c->stream));
    }
    CU(cudaMemcpyAsync(peaks_out, c->d_peaks, sizeof(PeakOut) * (size_t)nt, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return (found > trig_capacity) ? CBMF_WTRUNC : CBMF_OK;
}

extern "C" int cbmf_debug_td_template(cbmf_ctx* c, cbmf_template t, float* h_out)
{
    if (!c || !h_out) return CBMF_EINVAL;
    DeviceGuard g(c->device);
    int rc;
    if ((rc = grow(c, c->d_bank, c->bank_cap, 2))) return rc;
    if ((rc = grow(c, c->d_coef, c->coef_cap, 1))) return rc;
    if ((rc = grow(c, c->d_tcount, c->tcount_cap, 1))) return rc;
    if ((rc = td_alloc(c, 1, 1))) return rc;
    const size_t n = (size_t)c->n;
    if ((rc = grow_scratch(c, sizeof(float2) * n))) return rc;
    unsigned long long status[2] = {0ULL, (unsigned long long)NO_BAD_TEMPLATE};
    CU(cudaMemcpyAsync(c->d_cursor, status, sizeof(status), cudaMemcpyHostToDevice, c->stream));
    CU(cudaMemsetAsync(c->d_err, 0, sizeof(int), c->stream));
    CU(cudaMemcpyAsync(c->d_bank, &t, sizeof(t), cudaMemcpyHostToDevice, c->stream));
    if ((rc = td_setup(c, c->d_bank, 1, 0.f))) return rc;
    td_generate_kernel<<<dim3((unsigned)((n + 255) / 256), 1), 256, 0, c->stream>>>(c->d_td, c->d_tdU, (int)n, c->dt, 1.0f);
    CU(cudaGetLastError());
    td_copy_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->d_tdU, (float2*)c->d_scratch, (int)n);
    CU(cudaGetLastError());
    c->launches += 2;
    CU(cudaMemcpyAsync(status, c->d_cursor, sizeof(status), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaMemcpyAsync(h_out, c->d_scratch, sizeof(float2) * n, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return ((long long)status[1] != NO_BAD_TEMPLATE) ? CBMF_EINVAL : CBMF_OK;
}

// ======================================================================= diagnostics
// One template's coefficients into d_coef[0] (threshold 0).
static int setup_one(cbmf_ctx* c, cbmf_template t)
{
    int rc;
    if ((rc = grow(c, c->d_coef, c->coef_cap, 1))) return rc;
    if ((rc = grow(c, c->d_bank, c->bank_cap, 2))) return rc;
    CU(cudaMemsetAsync(c->d_err, 0, sizeof(int), c->stream));
    CU(cudaMemcpyAsync(c->d_bank, &t, sizeof(t), cudaMemcpyHostToDevice, c->stream));
    SetupArgs sa;
    sa.bank = c->d_bank; sa.prefix = c->d_prefix; sa.coef = c->d_coef; sa.n_templates = 1;
    sa.n_half = (int)(c->n / 2); sa.k_lo = c->k_lo; sa.n_over_fs = (double)c->n / c->fs; sa.df = c->df;
    sa.threshold = 0.f; sa.err_flag = c->d_err; sa.bad_idx = nullptr; sa.tcount = nullptr; sa.pn_half_order = c->pn_half_order;
    template_setup_kernel<<<1, 32, 0, c->stream>>>(sa);
    CU(cudaGetLastError());
    c->launches += 1;
    int err = 0;
    CU(cudaMemcpyAsync(&err, c->d_err, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return err ? CBMF_EINVAL : CBMF_OK;
}

extern "C" int cbmf_debug_snr_series(cbmf_ctx* c, cbmf_template t, float* snr_out, float* z_out)
{
    if (!c || !snr_out) return CBMF_EINVAL;
    if (!c->have_psd || !c->have_seg) return CBMF_ESTATE;
    DeviceGuard g(c->device);
    int rc;
    if ((rc = check_pending(c))) return rc;
    if ((rc = setup_one(c, t))) return rc;
    const size_t n = (size_t)c->n;
    if ((rc = grow_scratch(c, sizeof(float2) * n + sizeof(float) * n))) return rc;
    c2* z = (c2*)c->d_scratch;
    float* snr = (float*)(z + n);
    TemplCoef tc;
    CU(cudaMemcpyAsync(&tc, c->d_coef, sizeof(tc), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    P1Args a1; memset(&a1, 0, sizeof(a1));
    a1.w = c->d_w; a1.u = c->d_u; a1.lnk = c->d_lnk; a1.coef = c->d_coef; a1.Y = c->d_Y; a1.err_flag = c->d_err; a1.use_series = c->k_lo;
    CU(launch_p1<LOAD_GEN>(c, c->stream, a1, 1));
    P2Args a2; memset(&a2, 0, sizeof(a2));
    a2.Y = c->d_Y; a2.z_out = z;
    CU(launch_p2<EPI_STORE>(c, c->stream, a2, 1));
    snr_from_z_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>((const float2*)z, snr, n, tc.inv_sigma);
    CU(cudaGetLastError());
    c->launches += 3;
    CU(cudaMemcpyAsync(snr_out, snr, sizeof(float) * n, cudaMemcpyDeviceToHost, c->stream));
    if (z_out) CU(cudaMemcpyAsync(z_out, z, sizeof(float2) * n, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return CBMF_OK;
}

extern "C" int cbmf_debug_template(cbmf_ctx* c, cbmf_template t, float* h_out)
{
    if (!c || !h_out) return CBMF_EINVAL;
    if (!c->have_psd) return CBMF_ESTATE;                 // sigma comes from the PSD prefix table
    DeviceGuard g(c->device);
    int rc;
    if ((rc = check_pending(c))) return rc;
    if ((rc = setup_one(c, t))) return rc;
    // the PRODUCT generator (pass 1 of filter_bank) with unit weights, its inputs dumped instead of transformed
    const size_t n = (size_t)c->n, nh = n / 2;
    if ((rc = grow_scratch(c, sizeof(c2) * (nh + n) + sizeof(float2) * (nh + 1)))) return rc;
    c2* ones = (c2*)c->d_scratch;
    c2* q = ones + nh;
    float2* h = (float2*)(q + n);
    fill_ones_kernel<<<(unsigned)((nh + 255) / 256), 256, 0, c->stream>>>(ones, (int)nh);
    CU(cudaGetLastError());
    P1Args a1; memset(&a1, 0, sizeof(a1));
    a1.w = ones; a1.u = c->d_u; a1.lnk = c->d_lnk; a1.coef = c->d_coef; a1.Y = q; a1.err_flag = c->d_err; a1.use_series = c->k_lo;
    CU(launch_p1<LOAD_GEN_DUMP>(c, c->stream, a1, 1));
    debug_template_kernel<<<(unsigned)((nh + 1 + 255) / 256), 256, 0, c->stream>>>(q, h, (int)nh, c->df);
    CU(cudaGetLastError());
    c->launches += 3;
    CU(cudaMemcpyAsync(h_out, h, sizeof(float2) * (nh + 1), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return CBMF_OK;
}

extern "C" int cbmf_debug_ifft_dev(cbmf_ctx* c, const float* in_dev, float* out_dev, int64_t n, int64_t batch)
{
    if (!c || !in_dev || !out_dev || n != c->n || batch < 0) return CBMF_EINVAL;
    DeviceGuard g(c->device);
    const int sb = c->sub_batch;
    for (int64_t b0 = 0; b0 < batch; b0 += sb) {
        const int nb = (int)((batch - b0 < sb) ? (batch - b0) : sb);
        P1Args a1; memset(&a1, 0, sizeof(a1));
        a1.in_c = (const c2*)in_dev + (size_t)b0 * n; a1.Y = c->d_Y; a1.err_flag = c->d_err;
        CU(launch_p1_ifft(c, c->stream, a1, nb));
        P2Args a2; memset(&a2, 0, sizeof(a2));
        a2.Y = c->d_Y; a2.z_out = (c2*)out_dev + (size_t)b0 * n;
        CU(launch_p2_ifft(c, c->stream, a2, nb));
        c->launches += 2;
    }
    CU(cudaStreamSynchronize(c->stream));
    return CBMF_OK;
}

extern "C" int cbmf_debug_ifft(cbmf_ctx* c, const float* in, float* out, int64_t n, int64_t batch)
{
    if (!c || !in || !out || n != c->n || batch < 0) return CBMF_EINVAL;
    if (batch == 0) return CBMF_OK;
    DeviceGuard g(c->device);
    const size_t bytes = sizeof(c2) * (size_t)n * (size_t)batch;
    c2 *d_in = nullptr, *d_out = nullptr;
    CU(cudaMalloc(&d_in, bytes));
    cudaError_t e = cudaMalloc(&d_out, bytes);
    if (e != cudaSuccess) { cudaFree(d_in); return cuda_fail(c, e, "cudaMalloc"); }
    int rc = CBMF_OK;
    e = cudaMemcpyAsync(d_in, in, bytes, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) {
        rc = cbmf_debug_ifft_dev(c, (const float*)d_in, (float*)d_out, n, batch);
        if (rc == CBMF_OK) e = cudaMemcpyAsync(out, d_out, bytes, cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    }
    cudaFree(d_in); cudaFree(d_out);
    if (e != cudaSuccess) return cuda_fail(c, e, "cbmf_debug_ifft");
    return rc;
}

extern "C" int cbmf_debug_generate_dev(cbmf_ctx* c, const cbmf_template* bank_dev, int64_t nt, float* q_out_dev)
{
    if (!c || nt < 0 || (nt && (!bank_dev || !q_out_dev)) || nt > 65535) return CBMF_EINVAL;
    if (!c->have_psd || !c->have_seg) return CBMF_ESTATE;
    if (nt == 0) return CBMF_OK;
    DeviceGuard g(c->device);
    int rc;
    if ((rc = check_pending(c))) return rc;
    if ((rc = grow(c, c->d_coef, c->coef_cap, nt))) return rc;
    CU(cudaMemsetAsync(c->d_err, 0, sizeof(int), c->stream));
    SetupArgs sa;
    sa.bank = (const double*)bank_dev; sa.prefix = c->d_prefix; sa.coef = c->d_coef; sa.n_templates = (int)nt;
    sa.n_half = (int)(c->n / 2); sa.k_lo = c->k_lo; sa.n_over_fs = (double)c->n / c->fs; sa.df = c->df;
    sa.threshold = 0.f; sa.err_flag = c->d_err; sa.bad_idx = nullptr; sa.tcount = nullptr; sa.pn_half_order = c->pn_half_order;
    template_setup_kernel<<<(unsigned)((nt + 127) / 128), 128, 0, c->stream>>>(sa);
    CU(cudaGetLastError());
    const int nh = (int)(c->n / 2);
    int gx = (nh + 255) / 256; if (gx > 592) gx = 592;
    generate_only_kernel<<<dim3(gx, (unsigned)nt), 256, 0, c->stream>>>(c->d_w, c->d_u, c->d_lnk, c->d_coef, (c2*)q_out_dev, nh);
    CU(cudaGetLastError());
    c->launches += 2;
    int err = 0;
    CU(cudaMemcpyAsync(&err, c->d_err, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return err ? CBMF_EINVAL : CBMF_OK;
}

extern "C" int cbmf_debug_get_prefix(cbmf_ctx* c, double* p_out)
{
    if (!c || !p_out) return CBMF_EINVAL;
    if (!c->have_psd) return CBMF_ESTATE;
    DeviceGuard g(c->device);
    if (int r = check_pending(c)) return r;
    CU(cudaMemcpyAsync(p_out, c->d_prefix, sizeof(double) * (size_t)(c->n / 2), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return CBMF_OK;
}

extern "C" int cbmf_debug_get_weights(cbmf_ctx* c, float* w_out)
{
    if (!c || !w_out) return CBMF_EINVAL;
    if (!c->have_seg) return CBMF_ESTATE;
    DeviceGuard g(c->device);
    if (int r = check_pending(c)) return r;
    CU(cudaMemcpyAsync(w_out, c->d_w, sizeof(float2) * (size_t)(c->n / 2), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return CBMF_OK;
}

// ======================================================================= transform without allocation
// cbmf_ifft_noalloc_dev (include/cbmf.h): the stand-alone inverse FFT for callers that cannot allocate device memory
// where they need the transform -- guests of a framework whose allocator owns the GPU, real-time loops that must not
// hit the device-wide synchronisation of cudaMalloc / cudaFree, code running while a stream of the process is being
// captured.  Same kernels and the same split of n as cbmf_debug_ifft_dev, so the same numbers; the one difference is
// where the inter-pass buffer Y lives: in the array below, which is part of the library image, instead of in a
// context's cudaMalloc'ed d_Y.
namespace {

// Inter-pass buffer of the two-pass FFT: CBMF_NOALLOC_MAX_N packed complex floats = 8 MiB, held by every GPU that
// loads this library's device code until the process exits.  One array per GPU, shared by every call.
//
// In HOST code the name g_noalloc_Y is only a host-side handle of the symbol: its host "address" is not where the
// array lives on any GPU, and a kernel handed &g_noalloc_Y[0] from the host would fault (or, on a system whose GPUs
// can reach host memory, quietly scribble over host memory).  Host code therefore never passes the name to a
// kernel: noalloc_device() asks the runtime for the array's address ON THE CURRENT DEVICE (it differs from GPU to
// GPU) and the launches get that pointer.
static __device__ __align__(256) c2 g_noalloc_Y[CBMF_NOALLOC_MAX_N];

constexpr int NOALLOC_MAX_DEVICES = 64;
struct NoAllocDevice {
    c2* y = nullptr;                // device address of g_noalloc_Y on this GPU
    cbmf_ctx* shell = nullptr;      // host-only record the launch helpers want (SM count, shared-memory opt-ins): no device memory
};
NoAllocDevice g_noalloc_dev[NOALLOC_MAX_DEVICES];
std::mutex g_noalloc_mutex;         // guards the table above and the shell's fields

// Once per device, with that device current: the array's device address and the host-side record.  Runtime calls
// made: cudaGetSymbolAddress, cudaDeviceGetAttribute.  Nothing here allocates device memory.
int noalloc_device(int device, NoAllocDevice** out)
{
    NoAllocDevice& d = g_noalloc_dev[device];
    if (!d.y) {
        cbmf_ctx* c = nullptr;      // for CU()
        void* p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_noalloc_Y));
        if (!p) return CBMF_ECUDA;
        if (!d.shell) {
            d.shell = new (std::nothrow) cbmf_ctx();       // host heap only; lives as long as the process
            if (!d.shell) return CBMF_ENOMEM;
            d.shell->device = device;
        }
        CU(cudaDeviceGetAttribute(&d.shell->n_sm, cudaDevAttrMultiProcessorCount, device));
        d.y = (c2*)p;
    }
    *out = &d;
    return CBMF_OK;
}

}  // namespace

extern "C" int cbmf_ifft_noalloc_dev(int device, void* cuda_stream, const float* in_dev, float* out_dev,
                                     int64_t n, int64_t batch)
{
    if (batch < 0 || n < (int64_t(1) << 12) || (n & (n - 1)) != 0) return CBMF_EINVAL;
    if (n > (int64_t)CBMF_NOALLOC_MAX_N) return CBMF_ELIMIT;         // the fixed array holds one transform of at most this size
    if (device < 0 || device >= NOALLOC_MAX_DEVICES) return CBMF_EINVAL;
    if (batch > 0 && (!in_dev || !out_dev)) return CBMF_EINVAL;
    if (((uintptr_t)in_dev | (uintptr_t)out_dev) & 15) return CBMF_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess) { cudaGetLastError(); return CBMF_ECUDA; }
    if (device >= ndev) return CBMF_EINVAL;

    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    DeviceGuard g(device);
    if (!g.ok) { cudaGetLastError(); return CBMF_ECUDA; }
    NoAllocDevice* d = nullptr;
    if (int rc = noalloc_device(device, &d)) return rc;
    if (batch == 0) return CBMF_OK;

    cbmf_ctx* c = d->shell;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int lg = ilog2(n);
    c->n = n; c->log2n = lg;
    c->lg1 = lg / 2; c->lg2 = lg - c->lg1;                 // the split cbmf_create chooses for n <= 2^20
    // as many transforms per launch pair as the array holds; pairs follow each other on the stream, so pass 1 of
    // the next pair overwrites Y only after pass 2 of this one has read it
    const int64_t per_pair = (int64_t)CBMF_NOALLOC_MAX_N / n;
    for (int64_t b0 = 0; b0 < batch; b0 += per_pair) {
        const int nb = (int)std::min(per_pair, batch - b0);
        P1Args a1; memset(&a1, 0, sizeof(a1));
        a1.in_c = (const c2*)in_dev + (size_t)b0 * (size_t)n; a1.Y = d->y;
        CU(launch_p1<LOAD_CPLX>(c, st, a1, nb));
        P2Args a2; memset(&a2, 0, sizeof(a2));
        a2.Y = d->y; a2.z_out = (c2*)out_dev + (size_t)b0 * (size_t)n;
        CU(launch_p2<EPI_STORE>(c, st, a2, nb));
        c->launches += 2;
    }
    return CBMF_OK;
}

// ======================================================================= FP32 pipe probe (diagnostic)
extern "C" int cbmf_debug_fp32_peak(int device, double* tflops_ffma, double* tflops_ffma2)
{
    if (!tflops_ffma || !tflops_ffma2) return CBMF_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess) { cudaGetLastError(); return CBMF_ECUDA; }
    if (device < 0 || device >= ndev) return CBMF_EINVAL;
    const cudaError_t e = cbmf_probe::fp32_peak(device, tflops_ffma, tflops_ffma2);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cbmf_debug_fp32_peak");
    return CBMF_OK;
}

// ======================================================================= introspection
extern "C" int64_t cbmf_launch_count(const cbmf_ctx* c) { return c ? c->launches : -1; }

extern "C" int cbmf_last_pass_time(const cbmf_ctx* c, int which, double* ms_out, int64_t* launches_out)
{
    if (!c || which < 0 || which > 1) return CBMF_EINVAL;
    if (ms_out) *ms_out = c->last_ms[which];
    if (launches_out) *launches_out = c->last_launches[which];
    return CBMF_OK;
}

extern "C" int cbmf_debug_timeline(const cbmf_ctx* c, int which, float* start_end_ms, int64_t max_launches, int64_t* n_launches)
{
    if (!c || which < 0 || which > 1 || max_launches < 0 || (max_launches && !start_end_ms)) return CBMF_EINVAL;
    const int64_t n = (int64_t)c->timeline[which].size() / 2, k = n < max_launches ? n : max_launches;
    for (int64_t i = 0; i < 2 * k; ++i) start_end_ms[i] = c->timeline[which][(size_t)i];
    if (n_launches) *n_launches = n;
    return CBMF_OK;
}

extern "C" int cbmf_set_profiling(cbmf_ctx* c, int on)
{
    if (!c || on < 0 || on > 2) return CBMF_EINVAL;
    c->profiling = on;
    return CBMF_OK;
}

extern "C" const char* cbmf_strerror(int rc)
{
    switch (rc) {
        case CBMF_OK: return "success";
        case CBMF_EINVAL: return "invalid argument";
        case CBMF_ESTATE: return "call order: set_psd, then load_segment, then filter_bank";
        case CBMF_ECUDA: return "CUDA runtime error";
        case CBMF_ENOMEM: return "out of memory";
        case CBMF_ELIMIT: return "size exceeds the fixed scratch array of the no-allocation entry point";
        case CBMF_WTRUNC: return "trigger list truncated at trig_capacity";
        default: return "unknown code";
    }
}

extern "C" const char* cbmf_last_cuda_error(const cbmf_ctx* c) { return c ? c->cuda_err : ""; }

extern "C" const char* cbmf_version(void) { return "cbmf 0.1 (sm_100a)"; }
