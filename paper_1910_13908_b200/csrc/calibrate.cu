// sagecal_sage_calibrate: SAGE-EM over clusters with a block-diagonal Levenberg-Marquardt M-step, the whole loop
// enqueued on one stream with every decision taken on the device (SURVEY.md §8(a) rows 8a-3, 8a-5..8a-7,
// §8(c) A7-A8).  No device->host traffic, no synchronisation inside an interval.
#include <math.h>
#include <string.h>
#include "lm_pass.cuh"
#include "compress.cuh"

namespace sgc {

int corrupt_range(int N, int T, int F, int coh_format, const sagecal_c128* coh, const sagecal_c128* jones, int k0,
                  int k1, double sign, const sagecal_c128* vis_in, sagecal_c128* vis_out, cudaStream_t st);

thread_local int g_last_cuda_error = 0;

int num_sms() {
    static int cached[64] = {};
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) {
        (void)cudaGetLastError();
        return 148;  // B200; only reached without a device (workspace sizing on a CPU-only box)
    }
    if (cached[dev]) return cached[dev];
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
        (void)cudaGetLastError();
        return 148;
    }
    cached[dev] = n;
    return n;
}

// ---- LM control (8a-5): damping, 2x2 solves, accept/reject, all on device --------------------------------------
struct LmScalars {
    double phi;      // cost at the accepted Jones
    double phi_try;  // cost at the trial Jones (written by the pass)
    double mu, nu;   // Nielsen damping state
    double pred;     // predicted reduction of the pending trial step
    double pad[3];
};

constexpr int LM_THREADS = 256;

__device__ __forceinline__ double block_sum(double v, double* s_buf) {  // fixed-order tree, all threads get the sum
    const int tid = threadIdx.x;
    s_buf[tid] = v;
    __syncthreads();
    for (int o = LM_THREADS / 2; o > 0; o >>= 1) {
        if (tid < o) s_buf[tid] += s_buf[tid + o];
        __syncthreads();
    }
    const double r = s_buf[0];
    __syncthreads();
    return r;
}
__device__ __forceinline__ double block_max(double v, double* s_buf) {
    const int tid = threadIdx.x;
    s_buf[tid] = v;
    __syncthreads();
    for (int o = LM_THREADS / 2; o > 0; o >>= 1) {
        if (tid < o) s_buf[tid] = fmax(s_buf[tid], s_buf[tid + o]);
        __syncthreads();
    }
    const double r = s_buf[0];
    __syncthreads();
    return r;
}

// Direct mode's LM control (compressed mode: phase B of mstep_kernel; full Gauss-Newton: fgn_control_kernel).
// INIT:   (phi, G, M) were just evaluated at J.  mu = tau*max_p max(M_p00, M_p11), nu = 2; first trial step.
// !INIT:  (phi_try, G_try, M_try) were just evaluated at J_try.  rho test, accept/reject, damping update; next
//         trial step.  dJ_p = G_p (M_p + mu I)^-1, J_try = J + dJ, pred = sum_p Re tr(G_p^H dJ_p) + mu ||dJ_p||^2.
template <bool INIT>
__global__ void __launch_bounds__(LM_THREADS)
lm_step_kernel(int N, double tau, LmScalars* __restrict__ sc, sagecal_c128* __restrict__ J,
               sagecal_c128* __restrict__ G, sagecal_c128* __restrict__ M, const sagecal_c128* __restrict__ G_try,
               const sagecal_c128* __restrict__ M_try, sagecal_c128* __restrict__ J_try,
               double* __restrict__ cost_out, double* __restrict__ trace_out) {
    __shared__ double s_buf[LM_THREADS];
    const int tid = threadIdx.x;
    double phi = sc->phi, mu, nu;
    bool accept = false;
    if (INIT) {
        double mmax = 0.0;
        for (int p = tid; p < N; p += LM_THREADS) mmax = fmax(mmax, fmax(M[4 * p].re, M[4 * p + 3].re));
        mmax = block_max(mmax, s_buf);
        mu = tau * mmax;
        nu = 2.0;
    } else {
        const double phin = sc->phi_try, pred = sc->pred;
        mu = sc->mu; nu = sc->nu;
        const double rho = (phi - phin) / pred;
        accept = isfinite(phin) && isfinite(pred) && isfinite(rho) && pred > 0.0 && rho > 0.0;
        if (accept) {
            phi = phin;
            const double s = 2.0 * rho - 1.0;
            mu *= fmax(1.0 / 3.0, 1.0 - s * s * s);
            nu = 2.0;
        } else {
            mu *= nu;
            nu *= 2.0;
        }
    }
    if (!(mu >= 1e-300)) mu = 1e-300;
    if (mu > 1e300) mu = 1e300;
    if (nu > 0x1p60) nu = 0x1p60;

    double pred_part = 0.0;
    for (int p = tid; p < N; p += LM_THREADS) {
        cplx g[4], m[4], j[4];
#pragma unroll
        for (int i = 0; i < 4; i++) {
            if (accept) {
                g[i] = mk(G_try[4 * p + i].re, G_try[4 * p + i].im);
                m[i] = mk(M_try[4 * p + i].re, M_try[4 * p + i].im);
                j[i] = mk(J_try[4 * p + i].re, J_try[4 * p + i].im);
                G[4 * p + i].re = g[i].re; G[4 * p + i].im = g[i].im;
                M[4 * p + i].re = m[i].re; M[4 * p + i].im = m[i].im;
                J[4 * p + i].re = j[i].re; J[4 * p + i].im = j[i].im;
            } else {
                g[i] = mk(G[4 * p + i].re, G[4 * p + i].im);
                m[i] = mk(M[4 * p + i].re, M[4 * p + i].im);
                j[i] = mk(J[4 * p + i].re, J[4 * p + i].im);
            }
        }
        // (M_p + mu I)^-1 of the Hermitian 2x2 [[a, b], [conj b, d]]
        const double a = m[0].re + mu, d = m[3].re + mu;
        const cplx b = m[1];
        const double det = a * d - (b.re * b.re + b.im * b.im);
        const cplx inv[4] = {mk(d / det, 0.0), mk(-b.re / det, -b.im / det), mk(-b.re / det, b.im / det),
                             mk(a / det, 0.0)};
        cplx dj[4];
        dj[0] = cfma(g[1], inv[2], cmul(g[0], inv[0]));
        dj[1] = cfma(g[1], inv[3], cmul(g[0], inv[1]));
        dj[2] = cfma(g[3], inv[2], cmul(g[2], inv[0]));
        dj[3] = cfma(g[3], inv[3], cmul(g[2], inv[1]));
#pragma unroll
        for (int i = 0; i < 4; i++) {
            J_try[4 * p + i].re = j[i].re + dj[i].re;
            J_try[4 * p + i].im = j[i].im + dj[i].im;
            pred_part += g[i].re * dj[i].re + g[i].im * dj[i].im;
            pred_part += mu * (dj[i].re * dj[i].re + dj[i].im * dj[i].im);
        }
    }
    const double pred = block_sum(pred_part, s_buf);
    if (tid == 0) {
        sc->phi = phi; sc->mu = mu; sc->nu = nu; sc->pred = pred;
        if (cost_out) *cost_out = phi;
        if (trace_out) *trace_out = phi;
    }
}

// ---- ||R||_F^2 for cost_trace[0] -------------------------------------------------------------------------------
constexpr int NORM_THREADS = 256;
__global__ void __launch_bounds__(NORM_THREADS)
norm2_partial_kernel(const double* __restrict__ v, int64_t n4, double* __restrict__ partial) {
    __shared__ double s_buf[NORM_THREADS];
    double acc = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * NORM_THREADS + threadIdx.x; i < n4; i += (int64_t)gridDim.x * NORM_THREADS) {
        const d4 a = ldg256_stream(v + 4 * i);
        acc = fma(a.x, a.x, fma(a.y, a.y, fma(a.z, a.z, fma(a.w, a.w, acc))));
    }
    s_buf[threadIdx.x] = acc;
    __syncthreads();
    for (int o = NORM_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) s_buf[threadIdx.x] += s_buf[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = s_buf[0];
}
__global__ void __launch_bounds__(NORM_THREADS)
norm2_final_kernel(const double* __restrict__ partial, int n, double* __restrict__ out) {
    __shared__ double s_buf[NORM_THREADS];
    double acc = 0.0;
    for (int i = threadIdx.x; i < n; i += NORM_THREADS) acc += partial[i];
    s_buf[threadIdx.x] = acc;
    __syncthreads();
    for (int o = NORM_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) s_buf[threadIdx.x] += s_buf[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = s_buf[0];
}
constexpr int NORM_BLOCKS = 1024;

struct CalWorkspace {
    PassWorkspace pass;
    LmScalars* sc;
    sagecal_c128 *G, *M, *G_try, *M_try, *J_try;
    double* norm_partial;
    CompressWorkspace cw;
};
static size_t cal_extra_bytes(int N) {
    return 256 + 5 * round_up((size_t)N * 64, 256) + round_up(sizeof(double) * NORM_BLOCKS, 256);
}
static CalWorkspace carve_cal(const PassGeom& g, int K, bool scalar, void* ws) {
    CalWorkspace w;
    w.pass = carve_pass_workspace(g, ws);
    char* p = (char*)ws + pass_workspace_bytes(g);
    w.sc = (LmScalars*)p; p += 256;
    const size_t nj = round_up((size_t)g.N * 64, 256);
    w.G = (sagecal_c128*)p; p += nj;
    w.M = (sagecal_c128*)p; p += nj;
    w.G_try = (sagecal_c128*)p; p += nj;
    w.M_try = (sagecal_c128*)p; p += nj;
    w.J_try = (sagecal_c128*)p; p += nj;
    w.norm_partial = (double*)p; p += round_up(sizeof(double) * NORM_BLOCKS, 256);
    w.cw = carve_compress(g.N, K, scalar, p);
    return w;
}

template <bool INIT>
static int enqueue_step(int N, double tau, const CalWorkspace& w, sagecal_c128* Jk, double* cost_out, double* trace_out,
                        cudaStream_t st) {
    LaunchScope ls(KK_LMSTEP, st);
    lm_step_kernel<INIT><<<1, LM_THREADS, 0, st>>>(N, tau, w.sc, Jk, w.G, w.M, w.G_try, w.M_try, w.J_try, cost_out,
                                                  trace_out);
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}

}  // namespace sgc

using namespace sgc;

extern "C" const char* sagecal_strerror(int code) {
    switch (code) {
        case SAGECAL_OK: return "ok";
        case SAGECAL_EINVAL: return "invalid argument (shape, NULL or misaligned pointer, enum)";
        case SAGECAL_EWORKSPACE: return "workspace missing, misaligned or too small";
        case SAGECAL_ECUDA: return "CUDA call failed (see sagecal_last_cuda_error)";
        case SAGECAL_EUNSUPPORTED: return "valid request not implemented by this build";
        case SAGECAL_ESTATICLIMIT: return "request exceeds the fixed device scratch of a no-allocation entry point";
        default: return "unknown sagecal error code";
    }
}
extern "C" int sagecal_last_cuda_error(void) { return g_last_cuda_error; }
extern "C" const char* sagecal_version(void) { return "0.2.0"; }

extern "C" size_t sagecal_workspace_bytes(int what, int N, int T, int F, int K) {
    if (N < 2 || T < 1 || F < 1 || K < 0) return 0;
    const PassGeom g = make_pass_geom(N, T, F);
    switch (what) {
        case SAGECAL_WS_LM_PASS: return pass_workspace_bytes(g);
        // sized for either lm_mode and either coherency format (the general 2x2 statistics are the larger)
        case SAGECAL_WS_CALIBRATE: return pass_workspace_bytes(g) + cal_extra_bytes(N) + compress_workspace_bytes(N, K, false);
        case SAGECAL_WS_CALIBRATE_FULLGN:
            return pass_workspace_bytes(g) + cal_extra_bytes(N) + compress_workspace_bytes(N, K, false) + fullgn_workspace_bytes(N);
        default: return 0;
    }
}

// The residual is final time slot by time slot once the last write-back has passed: the host entry asks for that
// write-back in `final_chunks` ranges of time slots and is told after each (it starts the range's copy to the host on
// another stream while the next range is written).  The device entry runs it as one launch.
typedef int (*FinalChunkFn)(void* ctx, int t0, int t1);
static int sage_calibrate_core(int N, int T, int F, int K, const sagecal_c128* vis, int coh_format,
                               const sagecal_c128* coh, sagecal_c128* jones, sagecal_c128* residual, int n_em,
                               int n_lm, double tau, int lm_mode, double* cost_per_cluster, double* cost_trace,
                               void* workspace, size_t workspace_bytes, void* stream, int final_chunks,
                               FinalChunkFn after_chunk, void* after_ctx) {
    if (N < 2 || T < 1 || F < 1 || K < 0 || n_em < 0 || n_lm < 0) return SAGECAL_EINVAL;
    if (coh_format != SAGECAL_COH_FULL && coh_format != SAGECAL_COH_SCALAR) return SAGECAL_EINVAL;
    if (lm_mode != SAGECAL_LM_COMPRESSED && lm_mode != SAGECAL_LM_DIRECT && lm_mode != SAGECAL_LM_FULLGN && lm_mode != SAGECAL_LM_PERCLUSTER) return SAGECAL_EINVAL;
    // vis == NULL: `residual` already holds V - sum_k J_k C_k J_k^H at the start Jones (sagecal_predict_residual)
    if (!residual || vis == residual || (vis && !aligned(vis, 32)) || !aligned(residual, 32)) return SAGECAL_EINVAL;
    if (K > 0 && (!coh || !jones || !cost_per_cluster)) return SAGECAL_EINVAL;
    if (K > 0 && (!aligned(coh, coh_format == SAGECAL_COH_SCALAR ? 16 : 32) || !aligned(jones, 16))) return SAGECAL_EINVAL;
    if (!(tau > 0.0) || !isfinite(tau)) return SAGECAL_EINVAL;
    const PassGeom g = make_pass_geom(N, T, F);
    const size_t ws_base = sagecal_workspace_bytes(SAGECAL_WS_CALIBRATE, N, T, F, K);
    if (!workspace || !aligned(workspace, 256) ||
        workspace_bytes < (lm_mode == SAGECAL_LM_FULLGN ? sagecal_workspace_bytes(SAGECAL_WS_CALIBRATE_FULLGN, N, T, F, K) : ws_base))
        return SAGECAL_EWORKSPACE;
    void* fgn_ws = (char*)workspace + ws_base;
    const bool scalar = coh_format == SAGECAL_COH_SCALAR;
    const CalWorkspace w = carve_cal(g, K, scalar, workspace);
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t samples = (int64_t)T * g.B * F;
    const size_t cstride = scalar ? (size_t)samples : (size_t)samples * 4;
    int rc;
    if (final_chunks < 1) final_chunks = 1;
    if (final_chunks > T) final_chunks = T;
    const int tchunk = (T + final_chunks - 1) / final_chunks;
    const size_t rows_slot = (size_t)g.B * F;                 // samples per time slot
    auto whole = [&]() { return after_chunk ? after_chunk(after_ctx, 0, T) : SAGECAL_OK; };

    // R = V - sum_k J_k C_k J_k^H
    if (!vis) {
        // the initial residual came with the prediction
    } else if (K > 0) {
        if ((rc = corrupt_range(N, T, F, coh_format, coh, jones, 0, K, -1.0, vis, residual, st))) return rc;
    } else {
        SGC_CUDA(cudaMemcpyAsync(residual, vis, (size_t)samples * 64, cudaMemcpyDeviceToDevice, st));
    }
    if (cost_trace) {
        {
            LaunchScope ls(KK_NORM, st);
            norm2_partial_kernel<<<NORM_BLOCKS, NORM_THREADS, 0, st>>>((const double*)residual, samples * 2, w.norm_partial);
            SGC_LAUNCH_CHECK();
        }
        {
            LaunchScope ls(KK_NORM, st);
            norm2_final_kernel<<<1, NORM_THREADS, 0, st>>>(w.norm_partial, NORM_BLOCKS, cost_trace);
            SGC_LAUNCH_CHECK();
        }
    }
    if (K == 0 || n_em == 0) return whole();

    if (lm_mode == SAGECAL_LM_DIRECT) {
        // every LM evaluation streams the T*F samples of the cluster (rows 8a-3, 8a-4, 8a-6 as written)
        int it = 1;
        for (int em = 0; em < n_em; em++) {
            for (int k = 0; k < K; k++, it++) {
                const sagecal_c128* Ck = coh + (size_t)k * cstride;
                sagecal_c128* Jk = jones + (size_t)k * N * 4;
                double* tr = cost_trace ? cost_trace + it : nullptr;
                // E-step: x_k = R + J_k C_k J_k^H (in place: `residual` holds x_k during the M-step)
                if ((rc = corrupt_range(N, T, F, coh_format, coh, jones, k, k + 1, +1.0, residual, residual, st))) return rc;
                // M-step: n_lm trial steps of block-diagonal LM
                if ((rc = enqueue_pass(g, w.pass, residual, coh_format, Ck, Jk, &w.sc->phi, w.G, w.M, st))) return rc;
                if ((rc = enqueue_step<true>(N, tau, w, Jk, cost_per_cluster + k, tr, st))) return rc;
                for (int i = 0; i < n_lm; i++) {
                    if ((rc = enqueue_pass(g, w.pass, residual, coh_format, Ck, w.J_try, &w.sc->phi_try, w.G_try, w.M_try, st))) return rc;
                    if ((rc = enqueue_step<false>(N, tau, w, Jk, cost_per_cluster + k, tr, st))) return rc;
                }
                // R = x_k - J_k C_k J_k^H at the new J_k
                if ((rc = corrupt_range(N, T, F, coh_format, coh, jones, k, k + 1, -1.0, residual, residual, st))) return rc;
            }
        }
        return whole();
    }

    // compressed mode: `residual` always holds R; per (em, k) one streaming kernel writes back the
    // previous cluster and takes the statistics of the new residual against C_k (in the first EM iteration also the
    // gram Scc_k of the coherencies, kept for the later ones), then ONE cooperative kernel runs
    // the n_lm+1 evaluations and the LM control on the per-baseline statistics.  Statistics are re-centred every
    // SAGECAL_LM_RECENTRE trial steps.
    if (lm_mode == SAGECAL_LM_COMPRESSED && n_lm <= SAGECAL_LM_RECENTRE) {
        // cluster groups (wbgroup.cu): the write-back of GRP consecutive clusters is deferred and done in one pass
        // over R together with the statistics of the next GRP clusters; inside a group the statistics taken of the
        // stale residual are corrected per baseline through the cross grams X_ij of the coherencies.  An M-step is one
        // chunk here (n_lm <= SAGECAL_LM_RECENTRE); longer M-steps take the cluster-by-cluster loop below.
        const int64_t B = g.B;
        const size_t xgroup = (size_t)GRP_PAIRS * nxg(scalar) * B;       // doubles of cross grams per group
        const size_t srec = (size_t)nsrc(scalar) * B;
        int kp0 = 0, gp = 0, par = 0, it = 1;
        for (int em = 0; em < n_em; em++) {
            for (int k0 = 0; k0 < K; k0 += GRP) {
                const int gn = K - k0 < GRP ? K - k0 : GRP;
                double* Xgrp = w.cw.Xg + (size_t)(k0 / GRP) * xgroup;
                sagecal_c128* J0cur = w.cw.J0G + (size_t)par * GRP * N * 4;
                const sagecal_c128* J0prev = w.cw.J0G + (size_t)(par ^ 1) * GRP * N * 4;
                if ((rc = enqueue_wbgroup(N, T, F, coh_format, residual, coh, cstride, kp0, gp, J0prev, jones, k0, gn, w.cw.SrcG,
                                          em == 0 ? w.cw.Scc : nullptr, Xgrp, st))) return rc;
                for (int j = 0; j < gn; j++, it++) {
                    const int k = k0 + j;
                    sagecal_c128* Jk = jones + (size_t)k * N * 4;
                    sagecal_c128* J0 = J0cur + (size_t)j * N * 4;
                    const double* Scc_k = w.cw.Scc + (size_t)k * nscc(scalar) * B;
                    if (j > 0 && (rc = enqueue_groupfix(N, scalar, j, J0cur, jones + (size_t)k0 * N * 4,
                                                         w.cw.Scc + (size_t)(k - 1) * nscc(scalar) * B, Xgrp, w.cw.SrcG, st))) return rc;
                    CompressWorkspace cwj = w.cw;
                    cwj.Src = w.cw.SrcG + (size_t)j * srec;
                    if ((rc = enqueue_mstep(N, scalar, cwj, Scc_k, J0, Jk, n_lm, true, tau, cost_per_cluster + k,
                                            cost_trace ? cost_trace + it : nullptr, st))) return rc;
                }
                kp0 = k0; gp = gn; par ^= 1;
            }
        }
        // last write-back: the group solved last
        const sagecal_c128* J0prev = w.cw.J0G + (size_t)(par ^ 1) * GRP * N * 4;
        for (int t0 = 0; t0 < T; t0 += tchunk) {
            const int t1 = t0 + tchunk < T ? t0 + tchunk : T;
            const size_t off = (size_t)t0 * rows_slot;
            if ((rc = enqueue_wbgroup(N, t1 - t0, F, coh_format, residual + off * 4, coh + off * (scalar ? 1 : 4), cstride, kp0, gp,
                                      J0prev, jones, 0, 0, w.cw.SrcG, nullptr, nullptr, st))) return rc;
            if (after_chunk && (rc = after_chunk(after_ctx, t0, t1))) return rc;
        }
        return SAGECAL_OK;
    }

    // cluster by cluster: SAGECAL_LM_PERCLUSTER, SAGECAL_LM_FULLGN, and compressed M-steps longer than one chunk
    const sagecal_c128* Cprev = nullptr;      // cluster whose write-back is pending
    const sagecal_c128* Jprev = nullptr;
    const int64_t B = g.B;
    int par = 0;
    int it = 1;
    for (int em = 0; em < n_em; em++) {
        for (int k = 0; k < K; k++, it++) {
            const sagecal_c128* Ck = coh + (size_t)k * cstride;
            sagecal_c128* Jk = jones + (size_t)k * N * 4;
            double* Scc_k = w.cw.Scc + (size_t)k * nscc(scalar) * B;
            double* tr = cost_trace ? cost_trace + it : nullptr;
            int done = 0;
            do {
                sagecal_c128* J0 = w.cw.J0 + (size_t)par * N * 4;
                const sagecal_c128* J0prev = w.cw.J0 + (size_t)(par ^ 1) * N * 4;
                if ((rc = enqueue_wbstat(N, T, F, coh_format, residual, Cprev, J0prev, Jprev, Ck, w.cw.Src, em == 0 && done == 0 ? Scc_k : nullptr, st))) return rc;
                const int chunk = n_lm - done < SAGECAL_LM_RECENTRE ? n_lm - done : SAGECAL_LM_RECENTRE;
                if (lm_mode == SAGECAL_LM_FULLGN)
                    rc = enqueue_fullgn(N, scalar, w.cw, Scc_k, J0, Jk, chunk, done == 0, tau, cost_per_cluster + k, tr, fgn_ws, st);
                else
                    rc = enqueue_mstep(N, scalar, w.cw, Scc_k, J0, Jk, chunk, done == 0, tau, cost_per_cluster + k, tr, st);
                if (rc) return rc;
                done += chunk;
                Cprev = Ck; Jprev = Jk;
                par ^= 1;
            } while (done < n_lm);
        }
    }
    // last write-back: R -= dW c of the cluster solved last
    {
        const sagecal_c128* J0prev = w.cw.J0 + (size_t)(par ^ 1) * N * 4;
        for (int t0 = 0; t0 < T; t0 += tchunk) {
            const int t1 = t0 + tchunk < T ? t0 + tchunk : T;
            const size_t off = (size_t)t0 * rows_slot;
            if ((rc = enqueue_wbstat(N, t1 - t0, F, coh_format, residual + off * 4, Cprev ? Cprev + off * (scalar ? 1 : 4) : nullptr,
                                     J0prev, Jprev, nullptr, w.cw.Src, nullptr, st))) return rc;
            if (after_chunk && (rc = after_chunk(after_ctx, t0, t1))) return rc;
        }
    }
    return SAGECAL_OK;
}

extern "C" int sagecal_sage_calibrate(int N, int T, int F, int K, const sagecal_c128* vis, int coh_format,
                                      const sagecal_c128* coh, sagecal_c128* jones, sagecal_c128* residual, int n_em,
                                      int n_lm, double tau, int lm_mode, double* cost_per_cluster, double* cost_trace,
                                      void* workspace, size_t workspace_bytes, void* stream) {
    return sage_calibrate_core(N, T, F, K, vis, coh_format, coh, jones, residual, n_em, n_lm, tau, lm_mode,
                               cost_per_cluster, cost_trace, workspace, workspace_bytes, stream, 1, nullptr, nullptr);
}

// Per (host thread, device) helpers of the host entry, created once: TWO arenas the library keeps between calls
// (intervals arrive back to back; consecutive intervals alternate between them, so that one interval's output copies
// can still be in flight while the next is computed; plain cudaMalloc, no memory pool is touched), the copy
// stream and the events that order it against the caller's stream.
constexpr int HOST_FINAL_CHUNKS = 7;
struct HostCtx {
    bool ready = false;
    char* arena[2] = {nullptr, nullptr};
    size_t arena_bytes[2] = {0, 0};
    cudaStream_t cs = nullptr, cs_out = nullptr;        // host-to-device / device-to-host copy streams
    cudaEvent_t ev_vis = nullptr, ev_small = nullptr, ev_chunk[HOST_FINAL_CHUNKS + 1] = {};
    cudaEvent_t ev_done[2] = {};                        // end of the last two intervals (asynchronous entry)
    unsigned long long n_async = 0;
};
static int host_ctx(HostCtx** out) {
    static thread_local HostCtx ctx[64];
    int dev = 0;
    SGC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return SAGECAL_EUNSUPPORTED;
    HostCtx& c = ctx[dev];
    if (!c.ready) {
        SGC_CUDA(cudaStreamCreateWithFlags(&c.cs, cudaStreamNonBlocking));
        SGC_CUDA(cudaStreamCreateWithFlags(&c.cs_out, cudaStreamNonBlocking));
        SGC_CUDA(cudaEventCreateWithFlags(&c.ev_small, cudaEventDisableTiming));
        SGC_CUDA(cudaEventCreateWithFlags(&c.ev_done[0], cudaEventDisableTiming));
        SGC_CUDA(cudaEventCreateWithFlags(&c.ev_done[1], cudaEventDisableTiming));
        SGC_CUDA(cudaEventCreateWithFlags(&c.ev_vis, cudaEventDisableTiming));
        for (int i = 0; i <= HOST_FINAL_CHUNKS; i++) SGC_CUDA(cudaEventCreateWithFlags(&c.ev_chunk[i], cudaEventDisableTiming));
        c.ready = true;
    }
    *out = &c;
    return SAGECAL_OK;
}
// after a range of time slots of the residual is final: its copy to the host starts on the copy stream
struct HostFinal {
    HostCtx* c;
    cudaStream_t st;
    const char* dev_res;
    char* host_res;
    size_t bytes_slot;
    int n;
};
static int host_final_chunk(void* ctx, int t0, int t1) {
    HostFinal* h = (HostFinal*)ctx;
    if (!h->host_res) return SAGECAL_OK;
    cudaEvent_t ev = h->c->ev_chunk[h->n < HOST_FINAL_CHUNKS ? h->n : HOST_FINAL_CHUNKS];
    h->n++;
    SGC_CUDA(cudaEventRecord(ev, h->st));
    SGC_CUDA(cudaStreamWaitEvent(h->c->cs_out, ev, 0));
    SGC_CUDA(cudaMemcpyAsync(h->host_res + (size_t)t0 * h->bytes_slot, h->dev_res + (size_t)t0 * h->bytes_slot,
                             (size_t)(t1 - t0) * h->bytes_slot, cudaMemcpyDeviceToHost, h->c->cs_out));
    return SAGECAL_OK;
}

static int host_interval(int N, int T, int F, const double* freqs_host, double f0,
                         const double* uvw_host, int K, const int* cluster_offset_host,
                         const double* src_l, const double* src_m, const double* src_I,
                         const double* src_Q, const double* src_U, const double* src_V,
                         const double* src_alpha, int coh_format, const sagecal_c128* vis_host,
                         sagecal_c128* jones_host, sagecal_c128* residual_host, int n_em,
                         int n_lm, double tau, int lm_mode, double* cost_per_cluster_host,
                         double* cost_trace_host, void* stream, bool async) {
    if (N < 2 || T < 1 || F < 1 || K < 1 || n_em < 0 || n_lm < 0) return SAGECAL_EINVAL;
    if (!freqs_host || !uvw_host || !cluster_offset_host || !vis_host || !jones_host || !cost_per_cluster_host)
        return SAGECAL_EINVAL;
    if (coh_format != SAGECAL_COH_FULL && coh_format != SAGECAL_COH_SCALAR) return SAGECAL_EINVAL;
    const int S = cluster_offset_host[K];
    if (S < 0 || (S > 0 && (!src_l || !src_m || !src_I || !src_alpha))) return SAGECAL_EINVAL;
    const bool pol = src_Q || src_U || src_V;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t B = (int64_t)N * (N - 1) / 2, rows = (int64_t)T * B, samples = rows * F;
    const size_t vis_bytes = (size_t)samples * 64;
    const size_t coh_bytes = (size_t)K * samples * (coh_format == SAGECAL_COH_SCALAR ? 16 : 64);
    // unpolarised sky models predict in station form: room for the station phasors of as many time slots as fit 2 GiB
    const size_t ws_pred = pol ? sagecal_predict_workspace_bytes(F, S) : sagecal_predict_workspace_bytes_station(N, T, F, K, S);
    const size_t ws_cal = sagecal_workspace_bytes(lm_mode == SAGECAL_LM_FULLGN ? SAGECAL_WS_CALIBRATE_FULLGN : SAGECAL_WS_CALIBRATE,
                                                  N, T, F, K);
    const size_t ntrace = (size_t)n_em * K + 1;
    const size_t sS = round_up(sizeof(double) * (size_t)(S > 0 ? S : 1), 256);

    // one arena: uvw | 7 source columns | vis | residual | coh | jones | costs | trace | workspaces
    size_t off = 0;
    auto take = [&](size_t n) { size_t o = off; off += round_up(n, 256); return o; };
    const size_t o_uvw = take((size_t)rows * 24), o_src = take(7 * sS), o_vis = take(vis_bytes), o_res = take(vis_bytes),
                 o_coh = take(coh_bytes), o_jon = take((size_t)K * N * 64), o_cpc = take(sizeof(double) * K),
                 o_trc = take(sizeof(double) * ntrace), o_wsp = take(ws_pred), o_wsc = take(ws_cal);
    HostCtx* hc = nullptr;
    int rc = host_ctx(&hc);
    if (rc) return rc;
    // Consecutive intervals alternate between the two arenas; at most two are in flight: wait for the interval that
    // used this arena last (the one before the previous one).
    // The synchronous entry waits for everything in flight and always takes the first arena.
    const int slot = async ? (int)(hc->n_async & 1) : 0;
    SGC_CUDA(cudaEventSynchronize(hc->ev_done[slot]));
    if (!async) SGC_CUDA(cudaEventSynchronize(hc->ev_done[1]));
    if (hc->arena_bytes[slot] < off) {
        if (hc->arena[slot]) SGC_CUDA(cudaFree(hc->arena[slot]));
        hc->arena[slot] = nullptr; hc->arena_bytes[slot] = 0;
        SGC_CUDA(cudaMalloc((void**)&hc->arena[slot], off));
        hc->arena_bytes[slot] = off;
    }
    char* arena = hc->arena[slot];
    auto h2d_on = [&](cudaStream_t s, size_t o, const void* src, size_t n) {
        if (rc == SAGECAL_OK && src && n) {
            cudaError_t e = cudaMemcpyAsync(arena + o, src, n, cudaMemcpyHostToDevice, s);
            if (e != cudaSuccess) rc = cuda_fail(e);
        }
    };
    auto h2d = [&](size_t o, const void* src, size_t n) { h2d_on(st, o, src, n); };
    // the visibilities (the bulk of the input) travel on a second stream while `st` predicts the coherencies,
    // which need only uvw and the source table; `st` joins before the calibration reads them
    cudaStream_t cs = hc->cs;
    cudaEvent_t ev_vis = hc->ev_vis;
    h2d(o_uvw, uvw_host, (size_t)rows * 24);
    const double* cols[7] = {src_l, src_m, src_I, src_alpha, src_Q, src_U, src_V};
    double* dcol[7];
    for (int i = 0; i < 7; i++) {
        dcol[i] = (double*)(arena + o_src + i * sS);
        h2d(o_src + i * sS, cols[i], sizeof(double) * (size_t)S);
    }
    h2d(o_jon, jones_host, (size_t)K * N * 64);
    // issued after the small copies: the host-to-device copy engine serves its queue in order, and the prediction
    // must not wait behind 1.3 GB of visibilities
    h2d_on(cs, o_vis, vis_host, vis_bytes);
    if (rc == SAGECAL_OK) {
        cudaError_t e = cudaEventRecord(ev_vis, cs);
        if (e != cudaSuccess) rc = cuda_fail(e);
    }
    if (rc == SAGECAL_OK)
        rc = sagecal_predict_coherencies(N, T, F, freqs_host, f0, (const double*)(arena + o_uvw), K, cluster_offset_host,
                                         dcol[0], dcol[1], dcol[2], pol ? dcol[4] : nullptr, pol ? dcol[5] : nullptr,
                                         pol ? dcol[6] : nullptr, dcol[3], coh_format, (sagecal_c128*)(arena + o_coh), 0,
                                         arena + o_wsp, ws_pred, st);
    if (rc == SAGECAL_OK) {
        cudaError_t e = cudaStreamWaitEvent(st, ev_vis, 0);
        if (e != cudaSuccess) rc = cuda_fail(e);
    }
    // the last write-back runs in ranges of time slots; each range's copy to the host overlaps the next range's kernel
    HostFinal hf = {hc, st, arena + o_res, (char*)residual_host, (size_t)B * F * 64, 0};
    if (rc == SAGECAL_OK)
        rc = sage_calibrate_core(N, T, F, K, (const sagecal_c128*)(arena + o_vis), coh_format,
                                 (const sagecal_c128*)(arena + o_coh), (sagecal_c128*)(arena + o_jon),
                                 (sagecal_c128*)(arena + o_res), n_em, n_lm, tau, lm_mode, (double*)(arena + o_cpc),
                                 cost_trace_host ? (double*)(arena + o_trc) : nullptr, arena + o_wsc, ws_cal, st,
                                 HOST_FINAL_CHUNKS, host_final_chunk, &hf);
    // All device-to-host traffic goes on the output copy stream: a copy enqueued on `st` would queue behind the residual's
    // chunks on the copy engine and hold `st` (and with it the next interval's prediction) for their 25 ms.  The
    // interval is over for the arena when that stream has passed the last copy; `st` itself is free for the next
    // interval at once (the asynchronous entry).
    if (rc == SAGECAL_OK) {
        cudaError_t e = cudaEventRecord(hc->ev_small, st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(hc->cs_out, hc->ev_small, 0);
        if (e != cudaSuccess) rc = cuda_fail(e);
    }
    auto d2h = [&](void* dst, size_t o, size_t n) {
        if (rc == SAGECAL_OK && dst && n) {
            cudaError_t e = cudaMemcpyAsync(dst, arena + o, n, cudaMemcpyDeviceToHost, hc->cs_out);
            if (e != cudaSuccess) rc = cuda_fail(e);
        }
    };
    d2h(jones_host, o_jon, (size_t)K * N * 64);
    d2h(cost_per_cluster_host, o_cpc, sizeof(double) * K);
    d2h(cost_trace_host, o_trc, sizeof(double) * ntrace);
    if (rc == SAGECAL_OK) {
        cudaError_t e = cudaEventRecord(hc->ev_done[slot], hc->cs_out);
        if (e != cudaSuccess) rc = cuda_fail(e);
        if (rc == SAGECAL_OK && async) { hc->n_async++; return rc; }
    }
    // synchronous entry, or an error: wait for every stream that may touch the arena or the host buffers
    cudaError_t e0 = cudaStreamSynchronize(cs);
    cudaError_t e1 = cudaStreamSynchronize(hc->cs_out);
    cudaError_t e2 = cudaStreamSynchronize(st);
    if (rc == SAGECAL_OK && e0 != cudaSuccess) rc = cuda_fail(e0);
    if (rc == SAGECAL_OK && e1 != cudaSuccess) rc = cuda_fail(e1);
    if (rc == SAGECAL_OK && e2 != cudaSuccess) rc = cuda_fail(e2);
    return rc;
}

extern "C" int sagecal_calibrate_interval_host(int N, int T, int F, const double* freqs_host, double f0,
                                               const double* uvw_host, int K, const int* cluster_offset_host,
                                               const double* src_l, const double* src_m, const double* src_I,
                                               const double* src_Q, const double* src_U, const double* src_V,
                                               const double* src_alpha, int coh_format, const sagecal_c128* vis_host,
                                               sagecal_c128* jones_host, sagecal_c128* residual_host, int n_em,
                                               int n_lm, double tau, int lm_mode, double* cost_per_cluster_host,
                                               double* cost_trace_host, void* stream) {
    return host_interval(N, T, F, freqs_host, f0, uvw_host, K, cluster_offset_host, src_l, src_m, src_I, src_Q, src_U, src_V,
                         src_alpha, coh_format, vis_host, jones_host, residual_host, n_em, n_lm, tau, lm_mode,
                         cost_per_cluster_host, cost_trace_host, stream, false);
}

extern "C" int sagecal_calibrate_interval_host_async(int N, int T, int F, const double* freqs_host, double f0,
                                                     const double* uvw_host, int K, const int* cluster_offset_host,
                                                     const double* src_l, const double* src_m, const double* src_I,
                                                     const double* src_Q, const double* src_U, const double* src_V,
                                                     const double* src_alpha, int coh_format, const sagecal_c128* vis_host,
                                                     sagecal_c128* jones_host, sagecal_c128* residual_host, int n_em,
                                                     int n_lm, double tau, int lm_mode, double* cost_per_cluster_host,
                                                     double* cost_trace_host, void* stream) {
    return host_interval(N, T, F, freqs_host, f0, uvw_host, K, cluster_offset_host, src_l, src_m, src_I, src_Q, src_U, src_V,
                         src_alpha, coh_format, vis_host, jones_host, residual_host, n_em, n_lm, tau, lm_mode,
                         cost_per_cluster_host, cost_trace_host, stream, true);
}

extern "C" int sagecal_host_sync(void* stream) {
    HostCtx* hc = nullptr;
    int rc = host_ctx(&hc);
    if (rc) return rc;
    SGC_CUDA(cudaStreamSynchronize(hc->cs));
    SGC_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    SGC_CUDA(cudaStreamSynchronize(hc->cs_out));
    return SAGECAL_OK;
}

extern "C" int sagecal_host_trim(void* stream) {
    int rc = sagecal_host_sync(stream);
    if (rc) return rc;
    HostCtx* hc = nullptr;
    if ((rc = host_ctx(&hc))) return rc;
    for (int i = 0; i < 2; i++) {
        if (hc->arena[i]) SGC_CUDA(cudaFree(hc->arena[i]));
        hc->arena[i] = nullptr; hc->arena_bytes[i] = 0;
    }
    return SAGECAL_OK;
}
