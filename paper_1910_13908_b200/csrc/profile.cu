// Launch accounting and optional per-kernel CUDA-event timing (sagecal_launch_count, sagecal_profile_*).
// Measurement plumbing for bench.py's `roofline` and `gpu_launches` keys: every kernel launch of the library goes
// through a LaunchScope, which always counts it and, when timing of its kind is enabled, brackets it with an event
// pair recorded on the launching stream.  Nothing here touches the data path.
#include <atomic>
#include <mutex>
#include <vector>
#include "common.cuh"

namespace sgc {

static std::atomic<long long> g_launches[KK_COUNT];
static std::atomic<unsigned> g_timed_mask{0};
static std::mutex g_mu;
struct EvPair { cudaEvent_t a, b; int kind; };
static std::vector<EvPair> g_pairs;    // recorded since the last read
static std::vector<EvPair> g_free;     // event pairs ready for reuse

LaunchScope::LaunchScope(int kind_, cudaStream_t st_) : kind(kind_), st(st_), timed(false) {
    g_launches[kind].fetch_add(1, std::memory_order_relaxed);
    if (g_timed_mask.load(std::memory_order_relaxed) & (1u << kind)) {
        std::lock_guard<std::mutex> lk(g_mu);
        EvPair p;
        if (!g_free.empty()) { p = g_free.back(); g_free.pop_back(); }
        else if (cudaEventCreate(&p.a) != cudaSuccess || cudaEventCreate(&p.b) != cudaSuccess) { (void)cudaGetLastError(); return; }
        p.kind = kind;
        if (cudaEventRecord(p.a, st) != cudaSuccess) { (void)cudaGetLastError(); g_free.push_back(p); return; }
        g_pairs.push_back(p);
        end = p.b;                       // this scope's own end event (another host thread may append in between)
        timed = true;
    }
}
// a scope that encloses more than one kernel launch reports the others here (sagecal_launch_count counts kernels)
void count_more_launches(int kind, int n) { g_launches[kind].fetch_add(n, std::memory_order_relaxed); }
LaunchScope::~LaunchScope() {
    if (timed) (void)cudaEventRecord(end, st);
}

// FP64 issue peak, measured: 8 independent DFMA chains per thread, 1024 threads (8 warps per scheduler) on every SM.
// The roofline denominator of the ALU-bound kernels (predict, the M-step's baseline phase), taken in the same run
// and at the same clocks as the kernels it is compared with.
__global__ void __launch_bounds__(1024)
dfma_peak_kernel(double* out, int iters, double a, double b) {
    double x[8];
#pragma unroll
    for (int i = 0; i < 8; i++) x[i] = (double)threadIdx.x + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++) x[i] = fma(x[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += x[i];
    if (s == 12345.678) out[0] = s;      // never true: keeps the chains alive
}

// The same for the FP64 tensor-core path (DMMA m8n8k4, 256 FMAs per instruction): the denominator of the station-form
// prediction.  8 independent accumulator pairs per warp, 16 warps per SM.
__global__ void __launch_bounds__(512)
dmma_peak_kernel(double* out, int iters, double a, double b) {
    double d0[8], d1[8];
#pragma unroll
    for (int i = 0; i < 8; i++) { d0[i] = (double)threadIdx.x; d1[i] = (double)i; }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(d0[i]), "+d"(d1[i]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += d0[i] + d1[i];
    if (s == 12345.678) out[0] = s;      // never true: keeps the chains alive
}

}  // namespace sgc

using namespace sgc;

extern "C" int sagecal_profile_dmma_peak(int iters, double* fma_per_s_host, double* ms_host, void* stream) {
    if (iters < 1 || !fma_per_s_host) return SAGECAL_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int sms = num_sms();
    double* scratch = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    SGC_CUDA(cudaMalloc((void**)&scratch, 256));
    int rc = SAGECAL_OK;
    float best = 0.f;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = cuda_fail(cudaGetLastError());
    for (int rep = 0; rep < 4 && rc == SAGECAL_OK; rep++) {          // first repetition = warm-up
        cudaError_t e = cudaEventRecord(e0, st);
        dmma_peak_kernel<<<sms, 512, 0, st>>>(scratch, iters, 1.0000001, 1e-9);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventRecord(e1, st);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e != cudaSuccess) { rc = cuda_fail(e); break; }
        if (rep > 0 && (best == 0.f || ms < best)) best = ms;
    }
    if (e0) (void)cudaEventDestroy(e0);
    if (e1) (void)cudaEventDestroy(e1);
    (void)cudaFree(scratch);
    if (rc != SAGECAL_OK) return rc;
    *fma_per_s_host = (double)sms * 16.0 * 8.0 * 256.0 * iters / (best * 1e-3);     // warps x chains x FMAs per DMMA
    if (ms_host) *ms_host = best;
    return SAGECAL_OK;
}

extern "C" int sagecal_profile_dfma_peak(int iters, double* fma_per_s_host, double* ms_host, void* stream) {
    if (iters < 1 || !fma_per_s_host) return SAGECAL_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int sms = num_sms();
    double* scratch = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    SGC_CUDA(cudaMalloc((void**)&scratch, 256));
    int rc = SAGECAL_OK;
    float best = 0.f;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = cuda_fail(cudaGetLastError());
    for (int rep = 0; rep < 4 && rc == SAGECAL_OK; rep++) {          // first repetition = warm-up
        cudaError_t e = cudaEventRecord(e0, st);
        dfma_peak_kernel<<<sms, 1024, 0, st>>>(scratch, iters, 1.0000001, 1e-9);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventRecord(e1, st);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e != cudaSuccess) { rc = cuda_fail(e); break; }
        if (rep > 0 && (best == 0.f || ms < best)) best = ms;
    }
    if (e0) (void)cudaEventDestroy(e0);
    if (e1) (void)cudaEventDestroy(e1);
    (void)cudaFree(scratch);
    if (rc != SAGECAL_OK) return rc;
    *fma_per_s_host = (double)sms * 1024.0 * 8.0 * iters / (best * 1e-3);
    if (ms_host) *ms_host = best;
    return SAGECAL_OK;
}

extern "C" long long sagecal_launch_count(void) {
    long long n = 0;
    for (int k = 0; k < KK_COUNT; k++) n += g_launches[k].load();
    return n;
}

extern "C" int sagecal_kernel_kinds(void) { return KK_COUNT; }

extern "C" const char* sagecal_kernel_kind_name(int kind) {
    static const char* names[KK_COUNT] = {"predict_prep", "predict", "corrupt", "lm_pass", "lm_reduce", "lm_step", "norm2", "wbstat", "mstep", "fullgn", "rows", "groupfix"};
    return kind >= 0 && kind < KK_COUNT ? names[kind] : "?";
}

extern "C" int sagecal_profile_enable(unsigned kind_mask) {
    g_timed_mask.store(kind_mask & ((1u << KK_COUNT) - 1));
    return SAGECAL_OK;
}

extern "C" int sagecal_profile_read(double* ms_host, long long* timed_host, long long* launches_host) {
    std::lock_guard<std::mutex> lk(g_mu);
    for (int k = 0; k < KK_COUNT; k++) {
        if (ms_host) ms_host[k] = 0.0;
        if (timed_host) timed_host[k] = 0;
        if (launches_host) launches_host[k] = g_launches[k].load();
    }
    int rc = SAGECAL_OK;
    for (EvPair& p : g_pairs) {
        float ms = 0.f;
        cudaError_t e = cudaEventSynchronize(p.b);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, p.a, p.b);
        if (e != cudaSuccess) { rc = cuda_fail(e); (void)cudaGetLastError(); }
        else {
            if (ms_host) ms_host[p.kind] += (double)ms;
            if (timed_host) timed_host[p.kind]++;
        }
        g_free.push_back(p);
    }
    g_pairs.clear();
    return rc;
}
