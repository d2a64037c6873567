// Per-baseline statistics of the compressed M-step, fused with the previous cluster's write-back
// (SURVEY.md §8(a) rows 8a-3 / 8a-6 re-associated; formulas in compress.cuh).
//
//   wbstat:  R <- R - dW_prev c_prev   (write-back of the cluster just solved, dW_prev = W(J_prev) - W(J0_prev))
//            Src = sum_tf r c_next^H,  srr = sum_tf |r|^2   (statistics of the new residual for the next cluster)
//            Scc_next = sum_tf c_next c_next^H as well in the first EM iteration (it depends on the coherencies only
//            and is kept for the rest of the interval)
//
// HBM-bound streaming kernels: one thread owns one (baseline, channel) and walks the time slots, so at fixed t a
// warp reads 32 consecutive samples (2 KB, 256-bit loads); sums stay in registers over the time loop and are
// combined across the F lanes of a baseline with warp shuffles -- no atomics, fixed order.
#include "compress.cuh"

namespace sgc {

constexpr int WS_THREADS = 128;

__device__ __forceinline__ double group_sum(double v, int FP) {  // butterfly over the FP (power of two) lanes of a baseline
    for (int o = FP >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Scc += c c^H in the packed Hermitian layout of compress.cuh: 4 diagonal entries, then the 6 upper pairs
__device__ __forceinline__ void gram_add(const m22& c, double* acc) {
#pragma unroll
    for (int a = 0; a < 4; a++) acc[a] = cabs2(c.a[a], acc[a]);
    int pr = 0;
#pragma unroll
    for (int a = 0; a < 4; a++) {
#pragma unroll
        for (int c2 = a + 1; c2 < 4; c2++, pr++) {
            const cplx s = cfmac(c.a[a], c.a[c2], mk(acc[4 + 2 * pr], acc[5 + 2 * pr]));
            acc[4 + 2 * pr] = s.re;
            acc[5 + 2 * pr] = s.im;
        }
    }
}

// GRAM: also accumulate Scc of C_next (the first EM iteration; Scc depends on the coherencies only and is kept for
// the rest of the interval)
template <bool SCALAR, bool HAS_PREV, bool HAS_NEXT, bool GRAM>
__global__ void __launch_bounds__(WS_THREADS, SCALAR ? 4 : (GRAM ? 2 : 3))
wbstat_kernel(int N, int T, int F, int FP, int64_t B, sagecal_c128* R, const sagecal_c128* __restrict__ Cprev,
              const sagecal_c128* __restrict__ J0prev, const sagecal_c128* __restrict__ Jprev,
              const sagecal_c128* __restrict__ Cnext, double* __restrict__ Src, double* __restrict__ Scc) {
    constexpr int NW = SCALAR ? 4 : 16;                 // entries of dP / dW per baseline
    __shared__ cplx s_dw[HAS_PREV ? NW : 1][HAS_PREV ? WS_THREADS : 1];   // [entry][baseline of this CTA]
    const int tid = threadIdx.x;
    const int BL = WS_THREADS / FP;                      // baselines per CTA
    const int g = tid / FP, fl = tid - g * FP;
    const int64_t b = (int64_t)blockIdx.x * BL + g;

    if (HAS_PREV) {
        for (int e = tid; e < BL * NW; e += WS_THREADS) {
            const int bl = e / NW, w = e - bl * NW;
            const int64_t bb = (int64_t)blockIdx.x * BL + bl;
            cplx v = mk(0.0, 0.0);
            if (bb < B) {
                int p, q;
                bl_stations(N, bb, p, q);
                v = SCALAR ? dP_entry(J0prev, Jprev, p, q, w) : dW_entry(J0prev, Jprev, p, q, w >> 2, w & 3);
            }
            s_dw[w][bl] = v;
        }
        __syncthreads();
    }

    constexpr int NS = SCALAR ? 4 : 16;
    cplx S[HAS_NEXT ? NS : 1];
    double rr = 0.0;
#pragma unroll
    for (int i = 0; i < (HAS_NEXT ? NS : 1); i++) S[i] = mk(0.0, 0.0);
    constexpr int NG = GRAM ? (SCALAR ? NSCC_SCALAR : NSCC_FULL) : 1;
    double gacc[NG];
#pragma unroll
    for (int i = 0; i < NG; i++) gacc[i] = 0.0;

    if (b < B) {
        for (int f = fl; f < F; f += FP) {
            size_t idx = (size_t)b * F + f;
            const size_t step = (size_t)B * F;
#pragma unroll 1
            for (int t = 0; t < T; t++, idx += step) {
                m22 r;
                load_m22(R + idx * 4, r);
                if (HAS_PREV) {
                    if (SCALAR) {
                        const cplx cp = ldg128_stream(Cprev + idx);
#pragma unroll
                        for (int a = 0; a < 4; a++) r.a[a] = cfms(s_dw[a][g], cp, r.a[a]);
                    } else {
                        m22 cp;
                        load_m22_stream(Cprev + idx * 4, cp);
#pragma unroll
                        for (int a = 0; a < 4; a++) {
#pragma unroll
                            for (int c = 0; c < 4; c++) r.a[a] = cfms(s_dw[4 * a + c][g], cp.a[c], r.a[a]);
                        }
                    }
                    store_m22(R + idx * 4, r);
                }
                if (HAS_NEXT) {
                    if (SCALAR) {
                        const cplx cn = ldg128_stream(Cnext + idx);
#pragma unroll
                        for (int a = 0; a < 4; a++) S[a] = cfmac(r.a[a], cn, S[a]);
                        if (GRAM) gacc[0] = cabs2(cn, gacc[0]);
                    } else {
                        m22 cn;
                        load_m22_stream(Cnext + idx * 4, cn);
#pragma unroll
                        for (int a = 0; a < 4; a++) {
#pragma unroll
                            for (int c = 0; c < 4; c++) S[4 * a + c] = cfmac(r.a[a], cn.a[c], S[4 * a + c]);
                        }
                        if (GRAM) gram_add(cn, gacc);
                    }
                    rr = cabs2(r.a[3], cabs2(r.a[2], cabs2(r.a[1], cabs2(r.a[0], rr))));
                }
            }
        }
    }
    if (HAS_NEXT) {
        // all 32 lanes take part (lanes of a missing baseline carry zeros)
#pragma unroll
        for (int i = 0; i < NS; i++) {
            const double re = group_sum(S[i].re, FP), im = group_sum(S[i].im, FP);
            if (fl == 0 && b < B) {
                Src[(size_t)b * nsrc(SCALAR) + 2 * i] = re;
                Src[(size_t)b * nsrc(SCALAR) + 2 * i + 1] = im;
            }
        }
        rr = group_sum(rr, FP);
        if (fl == 0 && b < B) {
            Src[(size_t)b * nsrc(SCALAR) + 2 * NS] = rr;
            Src[(size_t)b * nsrc(SCALAR) + 2 * NS + 1] = 0.0;
        }
        if (GRAM) {
#pragma unroll
            for (int i = 0; i < NG; i++) {
                const double v = group_sum(gacc[i], FP);
                if (fl == 0 && b < B) Scc[(size_t)b * nscc(SCALAR) + i] = v;
            }
        }
    }
}

template <bool SCALAR>
static int launch_wbstat(int N, int T, int F, sagecal_c128* R, const sagecal_c128* Cprev, const sagecal_c128* J0prev,
                         const sagecal_c128* Jprev, const sagecal_c128* Cnext, double* Src, double* Scc, cudaStream_t st) {
    const int64_t B = (int64_t)N * (N - 1) / 2;
    const int FP = stat_group(F), BL = WS_THREADS / FP;
    const unsigned grid = (unsigned)((B + BL - 1) / BL);
    LaunchScope ls(KK_WBSTAT, st);
#define SGC_WB(P_, N_, G_) wbstat_kernel<SCALAR, P_, N_, G_><<<grid, WS_THREADS, 0, st>>>(N, T, F, FP, B, R, Cprev, J0prev, Jprev, Cnext, Src, Scc)
    if (Cprev && Cnext) { if (Scc) SGC_WB(true, true, true); else SGC_WB(true, true, false); }
    else if (Cprev) SGC_WB(true, false, false);
    else { if (Scc) SGC_WB(false, true, true); else SGC_WB(false, true, false); }
#undef SGC_WB
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}

int enqueue_wbstat(int N, int T, int F, int coh_format, sagecal_c128* R, const sagecal_c128* Cprev,
                   const sagecal_c128* J0prev, const sagecal_c128* Jprev, const sagecal_c128* Cnext, double* Src,
                   double* Scc_next, cudaStream_t st) {
    if (!Cprev && !Cnext) return SAGECAL_OK;
    return coh_format == SAGECAL_COH_SCALAR ? launch_wbstat<true>(N, T, F, R, Cprev, J0prev, Jprev, Cnext, Src, Scc_next, st)
                                            : launch_wbstat<false>(N, T, F, R, Cprev, J0prev, Jprev, Cnext, Src, Scc_next, st);
}

}  // namespace sgc
