// sagecal_corrupt_subtract: vis_out = vis_in + sign * sum_k J_{p,k} C_k J_{q,k}^H.
//
// HBM-bound, one pass over the visibilities: one thread owns one sample (64 B, two 256-bit accesses), walks the
// requested clusters in index order streaming C_k (no L1 allocation) while the per-station Jones come through the
// read-only L1 path (K*N*64 B, L2 resident).  In place is safe: a thread reads its sample before writing it.
#include "common.cuh"

namespace sgc {

constexpr int COR_THREADS = 256;

template <bool SCALAR, bool HAS_IN>
__global__ void __launch_bounds__(COR_THREADS)
corrupt_kernel(int N, int F, int64_t B, int64_t samples_per_slot, int64_t samples, int k0, int k1,
               const sagecal_c128* __restrict__ coh, const sagecal_c128* __restrict__ jones, double sign,
               const sagecal_c128* vis_in, sagecal_c128* vis_out) {
    const int64_t i = (int64_t)blockIdx.x * COR_THREADS + threadIdx.x;
    if (i >= samples) return;
    const int64_t b = (i % samples_per_slot) / F;
    int p, q;
    bl_stations(N, b, p, q);
    m22 acc;
    if (HAS_IN) load_m22(vis_in + 4 * i, acc);
    else { acc.a[0] = acc.a[1] = acc.a[2] = acc.a[3] = mk(0.0, 0.0); }

    const size_t cstride = SCALAR ? (size_t)samples : (size_t)samples * 4;
    const sagecal_c128* cp = coh + (size_t)k0 * cstride + (SCALAR ? (size_t)i : (size_t)i * 4);
#pragma unroll 2
    for (int k = k0; k < k1; k++, cp += cstride) {
        m22 Jp, Jq, model;
        load_jones(jones + ((size_t)k * N + p) * 4, Jp);
        load_jones(jones + ((size_t)k * N + q) * 4, Jq);
        if (SCALAR) {
            const cplx c = ldg128_stream(cp);
            m22 P;
            mmh(Jp, Jq, P);                        // J_p J_q^H
#pragma unroll
            for (int j = 0; j < 4; j++) model.a[j] = cmul(c, P.a[j]);
        } else {
            m22 C, T1;
            load_m22_stream(cp, C);
            mm(Jp, C, T1);                         // T1 = J_p C
            mmh(T1, Jq, model);                    // T1 J_q^H
        }
#pragma unroll
        for (int j = 0; j < 4; j++) {
            acc.a[j].re = fma(sign, model.a[j].re, acc.a[j].re);
            acc.a[j].im = fma(sign, model.a[j].im, acc.a[j].im);
        }
    }
    store_m22(vis_out + 4 * i, acc);
}

// Scalar coherencies, one thread per ROW (time slot, baseline) with all its channels: J_p J_q^H is formed once per
// (row, cluster) instead of once per sample (the per-sample form above spends ~60 FP64 instructions and two Jones loads
// on every 16-byte coherency and is FP64-bound: 7.5 ms for configs[4]'s 19.4 GB, 0.40 of the copy rate), and a channel
// costs 16 FMAs.  A lane reads and writes its own contiguous run (F x 16 B of coherencies per cluster, F x 64 B of
// visibilities) with 256-bit accesses: whole sectors.
constexpr int CORR_FT = 8;                 // channels per register tile
template <bool HAS_IN, bool EVENF>
__global__ void __launch_bounds__(128)
corrupt_scalar_rows_kernel(int N, int F, int64_t B, int64_t rows, int64_t samples, int k0, int k1,
                           const sagecal_c128* __restrict__ coh, const sagecal_c128* __restrict__ jones, double sign,
                           const sagecal_c128* vis_in, sagecal_c128* vis_out) {
    const int64_t r = (int64_t)blockIdx.x * 128 + threadIdx.x;
    if (r >= rows) return;
    int p, q;
    bl_stations(N, r % B, p, q);
    for (int c0 = 0; c0 < F; c0 += CORR_FT) {
        const int nf = min(CORR_FT, F - c0);
        m22 acc[CORR_FT];
#pragma unroll
        for (int c = 0; c < CORR_FT; c++) {
            if (HAS_IN && c < nf) load_m22(vis_in + ((size_t)r * F + c0 + c) * 4, acc[c]);
            else acc[c].a[0] = acc[c].a[1] = acc[c].a[2] = acc[c].a[3] = mk(0.0, 0.0);
        }
        const sagecal_c128* cp = coh + (size_t)k0 * samples + (size_t)r * F + c0;
#pragma unroll 2
        for (int k = k0; k < k1; k++, cp += samples) {
            m22 Jp, Jq, P;
            load_jones(jones + ((size_t)k * N + p) * 4, Jp);
            load_jones(jones + ((size_t)k * N + q) * 4, Jq);
            mmh(Jp, Jq, P);                        // J_p J_q^H
#pragma unroll
            for (int j = 0; j < 4; j++) { P.a[j].re *= sign; P.a[j].im *= sign; }
            cplx cv[CORR_FT];
            if (EVENF) {                           // (r F + c0) is even: 32-byte aligned pairs
#pragma unroll
                for (int c = 0; c < CORR_FT; c += 2) {
                    if (c < nf) {
                        const d4 v = ldg256_stream(cp + c);
                        cv[c] = mk(v.x, v.y); cv[c + 1] = mk(v.z, v.w);
                    }
                }
            } else {
#pragma unroll
                for (int c = 0; c < CORR_FT; c++)
                    if (c < nf) cv[c] = ldg128_stream(cp + c);
            }
#pragma unroll
            for (int c = 0; c < CORR_FT; c++) {
                if (c < nf) {
#pragma unroll
                    for (int j = 0; j < 4; j++) acc[c].a[j] = cfma(cv[c], P.a[j], acc[c].a[j]);
                }
            }
        }
#pragma unroll
        for (int c = 0; c < CORR_FT; c++)
            if (c < nf) store_m22(vis_out + ((size_t)r * F + c0 + c) * 4, acc[c]);
    }
}

// enqueue vis_out = vis_in + sign * sum_{k0<=k<k1} model_k
int corrupt_range(int N, int T, int F, int coh_format, const sagecal_c128* coh, const sagecal_c128* jones, int k0,
                  int k1, double sign, const sagecal_c128* vis_in, sagecal_c128* vis_out, cudaStream_t st) {
    const int64_t B = (int64_t)N * (N - 1) / 2;
    const int64_t samples = (int64_t)T * B * F;
    const unsigned grid = (unsigned)((samples + COR_THREADS - 1) / COR_THREADS);
    const bool scalar = coh_format == SAGECAL_COH_SCALAR;
    LaunchScope ls(KK_CORRUPT, st);
    if (scalar && F >= 2) {
        // one thread per row with all its channels (one J_p J_q^H per cluster)
        const int64_t rows = (int64_t)T * B;
        const unsigned g2 = (unsigned)((rows + 127) / 128);
        const bool evenf = (F & 1) == 0;
#define SGC_CSR(IN_, EV_) corrupt_scalar_rows_kernel<IN_, EV_><<<g2, 128, 0, st>>>(N, F, B, rows, samples, k0, k1, coh, jones, sign, vis_in, vis_out)
        if (vis_in) { if (evenf) SGC_CSR(true, true); else SGC_CSR(true, false); }
        else { if (evenf) SGC_CSR(false, true); else SGC_CSR(false, false); }
#undef SGC_CSR
    } else if (scalar) {
        if (vis_in) corrupt_kernel<true, true><<<grid, COR_THREADS, 0, st>>>(N, F, B, B * F, samples, k0, k1, coh, jones, sign, vis_in, vis_out);
        else corrupt_kernel<true, false><<<grid, COR_THREADS, 0, st>>>(N, F, B, B * F, samples, k0, k1, coh, jones, sign, vis_in, vis_out);
    } else {
        if (vis_in) corrupt_kernel<false, true><<<grid, COR_THREADS, 0, st>>>(N, F, B, B * F, samples, k0, k1, coh, jones, sign, vis_in, vis_out);
        else corrupt_kernel<false, false><<<grid, COR_THREADS, 0, st>>>(N, F, B, B * F, samples, k0, k1, coh, jones, sign, vis_in, vis_out);
    }
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}

}  // namespace sgc

using namespace sgc;

extern "C" int sagecal_corrupt_subtract(int N, int T, int F, int K, int coh_format, const sagecal_c128* coh,
                                        const sagecal_c128* jones, const uint8_t* cluster_mask_host, double sign,
                                        const sagecal_c128* vis_in, sagecal_c128* vis_out, void* stream) {
    if (N < 2 || T < 1 || F < 1 || K < 0) return SAGECAL_EINVAL;
    if (coh_format != SAGECAL_COH_FULL && coh_format != SAGECAL_COH_SCALAR) return SAGECAL_EINVAL;
    if (!vis_out || !aligned(vis_out, 32) || (vis_in && !aligned(vis_in, 32))) return SAGECAL_EINVAL;
    if (K > 0 && (!coh || !jones || !aligned(jones, 16))) return SAGECAL_EINVAL;
    if (K > 0 && !aligned(coh, coh_format == SAGECAL_COH_SCALAR ? 16 : 32)) return SAGECAL_EINVAL;
    if (!(sign == sign)) return SAGECAL_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t samples = (int64_t)T * ((int64_t)N * (N - 1) / 2) * F;

    // runs of consecutive selected clusters, in index order; the first run reads vis_in, later runs vis_out
    bool first = true;
    int k = 0;
    while (k < K) {
        if (cluster_mask_host && !cluster_mask_host[k]) { k++; continue; }
        int k1 = k + 1;
        while (k1 < K && (!cluster_mask_host || cluster_mask_host[k1])) k1++;
        int rc = corrupt_range(N, T, F, coh_format, coh, jones, k, k1, sign, first ? vis_in : vis_out, vis_out, st);
        if (rc) return rc;
        first = false;
        k = k1;
    }
    if (first) {  // nothing selected: vis_out = vis_in (or zeros)
        if (vis_in && vis_in != vis_out)
            SGC_CUDA(cudaMemcpyAsync(vis_out, vis_in, (size_t)samples * 64, cudaMemcpyDeviceToDevice, st));
        else if (!vis_in)
            SGC_CUDA(cudaMemsetAsync(vis_out, 0, (size_t)samples * 64, st));
    }
    return SAGECAL_OK;
}
