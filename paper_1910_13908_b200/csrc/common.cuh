// Shared device/host helpers of libsagecal_b200 (sm_100a).  Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "sagecal_b200.h"
#include "sagecal_b200_debug.h"

namespace sgc {

// ---- error plumbing -------------------------------------------------------------------------------------------
extern thread_local int g_last_cuda_error;
inline int cuda_fail(cudaError_t e) { g_last_cuda_error = (int)e; return SAGECAL_ECUDA; }
#define SGC_CUDA(call)                                   \
    do {                                                 \
        cudaError_t _e = (call);                         \
        if (_e != cudaSuccess) return sgc::cuda_fail(_e); \
    } while (0)
#define SGC_LAUNCH_CHECK() SGC_CUDA(cudaGetLastError())

inline bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }
inline size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
int num_sms();  // SM count of the current device (cached per device)

// ---- launch accounting and optional per-kernel CUDA-event timing (profile.cu; sagecal_profile_* in the ABI) ----
enum KernelKind { KK_PREP = 0, KK_PREDICT, KK_CORRUPT, KK_PASS, KK_REDUCE, KK_LMSTEP, KK_NORM, KK_WBSTAT, KK_MSTEP, KK_FULLGN, KK_ROWS, KK_GFIX, KK_COUNT };
// Brackets one kernel launch: counts it, and when timing of its kind is enabled records an event pair on `st`.
struct LaunchScope {
    int kind;
    cudaStream_t st;
    bool timed;
    cudaEvent_t end;
    LaunchScope(int kind, cudaStream_t st);
    ~LaunchScope();
};

void count_more_launches(int kind, int n);    // a LaunchScope counts one launch; the rest of its kernels go here

// ---- complex scalars and 2x2 matrices (row-major [XX, XY, YX, YY]) --------------------------------------------
struct __align__(16) cplx { double re, im; };
struct __align__(32) d4 { double x, y, z, w; };

__device__ __forceinline__ cplx mk(double re, double im) { cplx c; c.re = re; c.im = im; return c; }
// a*b
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
    return mk(fma(-a.im, b.im, a.re * b.re), fma(a.im, b.re, a.re * b.im));
}
// a*conj(b)
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) {
    return mk(fma(a.im, b.im, a.re * b.re), fma(a.im, b.re, -(a.re * b.im)));
}
// acc + a*b
__device__ __forceinline__ cplx cfma(cplx a, cplx b, cplx acc) {
    return mk(fma(-a.im, b.im, fma(a.re, b.re, acc.re)), fma(a.im, b.re, fma(a.re, b.im, acc.im)));
}
// acc - a*b
__device__ __forceinline__ cplx cfms(cplx a, cplx b, cplx acc) {
    return mk(fma(a.im, b.im, fma(-a.re, b.re, acc.re)), fma(-a.im, b.re, fma(-a.re, b.im, acc.im)));
}
// acc + a*conj(b)
__device__ __forceinline__ cplx cfmac(cplx a, cplx b, cplx acc) {
    return mk(fma(a.im, b.im, fma(a.re, b.re, acc.re)), fma(a.im, b.re, fma(-a.re, b.im, acc.im)));
}
// acc + conj(a)*b
__device__ __forceinline__ cplx cfmaca(cplx a, cplx b, cplx acc) {
    return mk(fma(a.im, b.im, fma(a.re, b.re, acc.re)), fma(-a.im, b.re, fma(a.re, b.im, acc.im)));
}
__device__ __forceinline__ double cabs2(cplx a, double acc) { return fma(a.im, a.im, fma(a.re, a.re, acc)); }

struct m22 { cplx a[4]; };

// o = a*b
__device__ __forceinline__ void mm(const m22& a, const m22& b, m22& o) {
    o.a[0] = cfma(a.a[1], b.a[2], cmul(a.a[0], b.a[0]));
    o.a[1] = cfma(a.a[1], b.a[3], cmul(a.a[0], b.a[1]));
    o.a[2] = cfma(a.a[3], b.a[2], cmul(a.a[2], b.a[0]));
    o.a[3] = cfma(a.a[3], b.a[3], cmul(a.a[2], b.a[1]));
}
// o = a*b^H
__device__ __forceinline__ void mmh(const m22& a, const m22& b, m22& o) {
    o.a[0] = cfmac(a.a[1], b.a[1], cmulc(a.a[0], b.a[0]));
    o.a[1] = cfmac(a.a[1], b.a[3], cmulc(a.a[0], b.a[2]));
    o.a[2] = cfmac(a.a[3], b.a[1], cmulc(a.a[2], b.a[0]));
    o.a[3] = cfmac(a.a[3], b.a[3], cmulc(a.a[2], b.a[2]));
}

// ---- 256-bit global accesses (sm_100+: LDG.E.256 / STG.E.256) -------------------------------------------------
__device__ __forceinline__ d4 ldg256_stream(const void* p) {  // read-once data: non-coherent, no L1 allocation
    d4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];"
                 : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ d4 ldg256(const void* p) {  // coherent (buffer may be written by the same kernel)
    d4 r;
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];"
                 : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void stg256(void* p, double x, double y, double z, double w) {
    asm volatile("st.global.v4.f64 [%4], {%0,%1,%2,%3};" ::"d"(x), "d"(y), "d"(z), "d"(w), "l"(p) : "memory");
}
__device__ __forceinline__ cplx ldg128_stream(const void* p) {
    cplx r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(r.re), "=d"(r.im) : "l"(p));
    return r;
}
// one 2x2 sample = 64 B = two 256-bit loads
__device__ __forceinline__ void load_m22_stream(const sagecal_c128* p, m22& o) {
    d4 lo = ldg256_stream(p), hi = ldg256_stream(p + 2);
    o.a[0] = mk(lo.x, lo.y); o.a[1] = mk(lo.z, lo.w); o.a[2] = mk(hi.x, hi.y); o.a[3] = mk(hi.z, hi.w);
}
__device__ __forceinline__ void load_m22(const sagecal_c128* p, m22& o) {
    d4 lo = ldg256(p), hi = ldg256(p + 2);
    o.a[0] = mk(lo.x, lo.y); o.a[1] = mk(lo.z, lo.w); o.a[2] = mk(hi.x, hi.y); o.a[3] = mk(hi.z, hi.w);
}
__device__ __forceinline__ void store_m22(sagecal_c128* p, const m22& v) {
    stg256(p, v.a[0].re, v.a[0].im, v.a[1].re, v.a[1].im);
    stg256(p + 2, v.a[2].re, v.a[2].im, v.a[3].re, v.a[3].im);
}
// Jones matrices are small, re-read by every thread: default (L1-allocating) read-only path
__device__ __forceinline__ void load_jones(const sagecal_c128* p, m22& o) {
    const double2* q = reinterpret_cast<const double2*>(p);
#pragma unroll
    for (int i = 0; i < 4; i++) { double2 v = __ldg(q + i); o.a[i] = mk(v.x, v.y); }
}

// ---- canonical baseline order: b(p,q) = p*N - p(p+1)/2 + (q-p-1), p<q ----------------------------------------
__host__ __device__ __forceinline__ int64_t row_start(int N, int p) {  // b(p, p+1)
    return (int64_t)p * N - (int64_t)p * (p + 1) / 2;
}
__host__ __device__ __forceinline__ int64_t bl_index(int N, int p, int q) { return row_start(N, p) + (q - p - 1); }
__device__ __forceinline__ void bl_stations(int N, int64_t b, int& p, int& q) {
    // invert b = p*N - p(p+1)/2 + (q-p-1): float estimate + exact integer fix-up
    float tn = 2.0f * (float)N - 1.0f;
    float disc = fmaxf(tn * tn - 8.0f * (float)b, 0.0f);
    int pp = (int)((tn - sqrtf(disc)) * 0.5f);
    pp = max(0, min(pp, N - 2));
    while (pp > 0 && row_start(N, pp) > b) pp--;
    while (pp < N - 2 && row_start(N, pp + 1) <= b) pp++;
    p = pp;
    q = pp + 1 + (int)(b - row_start(N, pp));
}

}  // namespace sgc
