// Cluster-group form of the compressed M-step's streaming kernel (DESIGN.md §5.5 "cluster groups").
//
// wbstat.cu moves 256 B per sample and cluster: R read and written, C_prev, C_next.  The statistics are linear in R,
// so R need not be current when they are taken: for a group of GRP consecutive clusters
//
//   wbgroup:   R <- R - sum_{i in previous group} dW_i c_i          (ONE read and ONE write of R per group)
//              Src_j = sum_tf r c_j^H for every j in the next group, srr = sum_tf |r|^2
//   groupfix:  right before cluster j of the group is solved, with the clusters i < j of the group solved so far
//              Src_j <- Src_j - sum_i dW_i X_ij,  X_ij = sum_tf c_i c_j^H  (r' = r - dW_i c_i  =>  r' c_j^H = r c_j^H - dW_i c_i c_j^H)
//              srr_j = srr_{j-1} - Re tr(dW_{j-1}^H (Src_{j-1} + Sec_{j-1}))   (the cost per baseline after j-1's update)
//   cross grams X_ij and Scc_i of a group: once per interval (they depend on the coherencies only), by the GRAM arm of
//              wbgroup in the first EM iteration
//
// (2 + 2 GRP) x 64 B per sample and group instead of GRP x 256 B: 160 B instead of 256 B per cluster at GRP = 4
// (2x2 coherencies; 64 B instead of 160 B with scalar coherencies).  Nothing is approximated; the LM trajectory is the
// same to rounding.
//
// Scalar coherencies: plain FP64 FMAs, one thread per (baseline, channel) sample as in wbstat.cu (8 accumulators per
// cluster; the cross grams ride along in the first EM iteration); sums over the channel lanes of a baseline by warp shuffles.  2x2 coherencies: the FP64 tensor cores, one
// warp per baseline (below).  Fixed order, no atomics.
#include "compress.cuh"

namespace sgc {

constexpr int WG_THREADS = 128;

// sum over n consecutive lanes (n a power of two)
__device__ __forceinline__ double lanes_sum(double v, int n) {
    for (int o = n >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- scalar coherencies: write-back of the previous group + statistics of the next group ------------------------------
// GRAM (first EM iteration): also s2_i = sum |c_i|^2 and x_ij = sum c_i conj(c_j) (i < j) of the next group, from the
// coherency samples the statistics load anyway.
template <int GP, int GN, bool GRAM>
__global__ void __launch_bounds__(WG_THREADS, 3)
wbgroup_scalar_kernel(int N, int T, int F, int FP, int64_t B, sagecal_c128* R, const sagecal_c128* __restrict__ coh,
                      size_t cstride, int kp0, const sagecal_c128* __restrict__ J0prev,
                      const sagecal_c128* __restrict__ jones, int kn0, double* __restrict__ SrcG,
                      double* __restrict__ Scc, double* __restrict__ Xg) {
    constexpr int GPn = GP > 0 ? GP : 1, GNn = GN > 0 ? GN : 1;
    __shared__ cplx s_dp[GPn][4][WG_THREADS];            // dP_i[a] per [cluster][entry][baseline of this CTA]
    const int tid = threadIdx.x;
    const int BL = WG_THREADS / FP;                      // baselines per CTA
    const int g = tid / FP, fl = tid - g * FP;
    const int64_t b = (int64_t)blockIdx.x * BL + g;

    if (GP > 0) {
        for (int e = tid; e < BL * 4 * GP; e += WG_THREADS) {
            const int i = e / (BL * 4), rem = e - i * (BL * 4);
            const int bl = rem >> 2, w = rem & 3;
            const int64_t bb = (int64_t)blockIdx.x * BL + bl;
            cplx v = mk(0.0, 0.0);
            if (bb < B) {
                int p, q;
                bl_stations(N, bb, p, q);
                v = dP_entry(J0prev + (size_t)i * N * 4, jones + (size_t)(kp0 + i) * N * 4, p, q, w);
            }
            s_dp[i][w][bl] = v;
        }
        __syncthreads();
    }

    cplx S[GNn][4];                                      // Sr_j[a]
#pragma unroll
    for (int j = 0; j < GNn; j++)
#pragma unroll
        for (int a = 0; a < 4; a++) S[j][a] = mk(0.0, 0.0);
    double rr = 0.0;
    constexpr int NP = GRAM ? GNn * (GNn + 1) / 2 : 1;
    cplx X[NP];
#pragma unroll
    for (int n = 0; n < NP; n++) X[n] = mk(0.0, 0.0);

    if (b < B) {
        const sagecal_c128* cprev = coh + (size_t)kp0 * cstride;
        const sagecal_c128* cnext = coh + (size_t)kn0 * cstride;
        const size_t step = (size_t)B * F;
        for (int f = fl; f < F; f += FP) {
            size_t idx = (size_t)b * F + f;
#pragma unroll 1
            for (int t = 0; t < T; t++, idx += step) {
                cplx cp[GPn], cn[GNn];
                m22 r;
                load_m22(R + idx * 4, r);
#pragma unroll
                for (int i = 0; i < GP; i++) cp[i] = ldg128_stream(cprev + (size_t)i * cstride + idx);
#pragma unroll
                for (int j = 0; j < GN; j++) cn[j] = ldg128_stream(cnext + (size_t)j * cstride + idx);
#pragma unroll
                for (int i = 0; i < GP; i++)
#pragma unroll
                    for (int a = 0; a < 4; a++) r.a[a] = cfms(s_dp[i][a][g], cp[i], r.a[a]);
                if (GP > 0) store_m22(R + idx * 4, r);
#pragma unroll
                for (int j = 0; j < GN; j++)
#pragma unroll
                    for (int a = 0; a < 4; a++) S[j][a] = cfmac(r.a[a], cn[j], S[j][a]);
                rr = cabs2(r.a[3], cabs2(r.a[2], cabs2(r.a[1], cabs2(r.a[0], rr))));
                if (GRAM) {
                    int n = 0;
#pragma unroll
                    for (int i = 0; i < GN; i++)
#pragma unroll
                        for (int j = i; j < GN; j++, n++) X[n] = cfmac(cn[i], cn[j], X[n]);
                }
            }
        }
    }
    if (GRAM) {
        const bool writer = fl == 0 && b < B;
        const size_t bb = b < B ? (size_t)b : 0;
        int n = 0;
#pragma unroll
        for (int i = 0; i < GN; i++)
#pragma unroll
            for (int j = i; j < GN; j++, n++) {
                const double re = lanes_sum(X[n].re, FP), im = lanes_sum(X[n].im, FP);
                if (!writer) continue;
                if (i == j) Scc[((size_t)(kn0 + i) * B + bb) * NSCC_SCALAR] = re;
                else {
                    double* o = Xg + ((size_t)grp_pair(i, j) * B + bb) * NX_SCALAR;
                    o[0] = re;
                    o[1] = im;
                }
            }
    }
    if (GN > 0) {
        const bool writer = fl == 0 && b < B;
        const size_t bb = b < B ? (size_t)b : 0;
#pragma unroll
        for (int j = 0; j < GN; j++) {
            double* rec = SrcG + ((size_t)j * B + bb) * NSRC_SCALAR;
#pragma unroll
            for (int a = 0; a < 4; a++) {
                const double re = lanes_sum(S[j][a].re, FP), im = lanes_sum(S[j][a].im, FP);
                if (writer) { rec[2 * a] = re; rec[2 * a + 1] = im; }
            }
        }
        rr = lanes_sum(rr, FP);
        if (writer) {
#pragma unroll
            for (int j = 0; j < GN; j++) {
                double* rec = SrcG + ((size_t)j * B + bb) * NSRC_SCALAR;
                rec[NSRC_SCALAR - 2] = rr;        // meaningful for j = 0; groupfix rewrites it for the later clusters
                rec[NSRC_SCALAR - 1] = 0.0;
            }
        }
    }
}

// ---- 2x2 coherencies on the FP64 tensor cores (DMMA m8n8k4) ----------------------------------------------------------
// The statistics are the one dense contraction of this path: per baseline Src_j = R^T conj(C_j) is a (4 x TF)(TF x 4)
// complex product, TF = T*F samples.  In real form a sample is 8 doubles (position g = 2a + ri), and
//   stats     : D_j[g][n] += sum_k r'[sample k][g] * c_j[sample k][n]          (8 x 8 += (8 x 4)(4 x 8), k = 4 samples)
//   write-back: r'[g][sample n] = r[g][sample n] + sum_k (-W_i)[g][k] c_i[sample n][k]   (k = 8 positions, two k-steps;
//               W_i = real 8 x 8 form of dW_i, constant per baseline: 2 registers per lane and cluster)
// One warp owns one baseline and walks its TF samples 8 at a time.  The fragment layouts line up so that nothing is
// shuffled: the write-back's D fragment (row g, samples 2j and 2j+1, j = lane & 3) IS the A fragment of the statistics
// if k-step s takes sample 2j + s, and the B fragments are 8-byte loads straight from global memory (a warp reads the 512
// contiguous bytes of 8 samples in two instructions).  Per 8 samples and group: 18 loads, 2 stores, 16 DMMA -- against
// ~370 instructions in the DFMA form; accumulators 2 doubles per lane and cluster.  Src = (rr + ii) + i (ir - ri) is
// combined once per baseline with the partner lane (lane ^ 4) that holds the other real/imaginary row.
__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__device__ __forceinline__ double ldg64_stream(const double* p) {
    double r;
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(r) : "l"(p));
    return r;
}
__device__ __forceinline__ double ld64(const double* p) {
    double r;
    asm volatile("ld.global.f64 %0, [%1];" : "=d"(r) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st64(double* p, double v) { asm volatile("st.global.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory"); }

constexpr int MMA_WARPS = 4;
// index (in samples) of sample m = t*F + f of baseline b, or -1 past the end
template <bool F8>
__host__ __device__ __forceinline__ int64_t sample_index(int m, int TF, int F, int64_t B, int64_t b) {
    if (m >= TF) return -1;
    if (F8) return ((int64_t)(m >> 3) * B + b) * 8 + (m & 7);
    const int t = m / F;
    return ((int64_t)t * B + b) * F + (m - t * F);
}

// GRAM (first EM iteration): also X_ij[a][c] = sum c_i[a] conj(c_j[c]) (i < j) and Scc_i of the next group -- the same
// contraction with both operands coherencies.  The B fragments of the statistics (position lane >> 2 of sample
// 2 (lane & 3) + s) serve as A for their cluster's rows and as B for its columns, so the cross grams cost no load at
// all, only GN (GN + 1) more DMMA per 8 samples.
template <int GP, int GN, bool F8, bool GRAM>
__global__ void __launch_bounds__(32 * MMA_WARPS, GRAM ? 4 : 5)
wbgroup_mma_kernel(int N, int T, int F, int64_t B, sagecal_c128* R_, const sagecal_c128* __restrict__ coh_,
                   size_t cstride, int kp0, const sagecal_c128* __restrict__ J0prev,
                   const sagecal_c128* __restrict__ jones, int kn0, double* __restrict__ SrcG,
                   double* __restrict__ Scc, double* __restrict__ Xg) {
    constexpr int GPn = GP > 0 ? GP : 1, GNn = GN > 0 ? GN : 1;
    const int lane = threadIdx.x & 31;
    const int64_t b = (int64_t)blockIdx.x * MMA_WARPS + (threadIdx.x >> 5);
    if (b >= B) return;                                   // whole warps leave together
    const int g = lane >> 2, j = lane & 3;
    double* R = reinterpret_cast<double*>(R_);
    const double* cprev = reinterpret_cast<const double*>(coh_ + (size_t)kp0 * cstride);
    const double* cnext = reinterpret_cast<const double*>(coh_ + (size_t)kn0 * cstride);
    const size_t cs = cstride * 2;                        // doubles per cluster

    double Aw[GPn][2];                                    // A fragments of -W_i: row g, column 4s + j
    if (GP > 0) {
        int p, q;
        bl_stations(N, b, p, q);
        const int a = g >> 1, ri = g & 1;
#pragma unroll
        for (int i = 0; i < GP; i++) {
#pragma unroll
            for (int s = 0; s < 2; s++) {
                const int kk = 4 * s + j, c = kk >> 1, ri2 = kk & 1;
                const cplx w = dW_entry(J0prev + (size_t)i * N * 4, jones + (size_t)(kp0 + i) * N * 4, p, q, a, c);
                // (w c).re = w.re c.re - w.im c.im,  (w c).im = w.im c.re + w.re c.im
                Aw[i][s] = -(ri == ri2 ? w.re : (ri ? w.im : -w.im));
            }
        }
    }
    double D[GNn][2];
#pragma unroll
    for (int jn = 0; jn < GNn; jn++) D[jn][0] = D[jn][1] = 0.0;
    double rr = 0.0;
    constexpr int NP = GRAM ? GNn * (GNn + 1) / 2 : 1;
    double X[NP][2];
#pragma unroll
    for (int n = 0; n < NP; n++) X[n][0] = X[n][1] = 0.0;

    const int TF = T * F;
#pragma unroll 1
    for (int m0 = 0; m0 < TF; m0 += 8) {
        const int64_t in = sample_index<F8>(m0 + g, TF, F, B, b);             // sample n = g (B fragments of the write-back)
        const int64_t i0 = sample_index<F8>(m0 + 2 * j, TF, F, B, b);         // samples 2j, 2j + 1 (C / D / A fragments)
        const int64_t i1 = sample_index<F8>(m0 + 2 * j + 1, TF, F, B, b);
        double c0 = i0 >= 0 ? ld64(R + i0 * 8 + g) : 0.0;
        double c1 = i1 >= 0 ? ld64(R + i1 * 8 + g) : 0.0;
        double bp[GPn][2], bn[GNn][2];
#pragma unroll
        for (int i = 0; i < GP; i++) {
            bp[i][0] = in >= 0 ? ldg64_stream(cprev + i * cs + in * 8 + j) : 0.0;
            bp[i][1] = in >= 0 ? ldg64_stream(cprev + i * cs + in * 8 + 4 + j) : 0.0;
        }
#pragma unroll
        for (int jn = 0; jn < GN; jn++) {
            bn[jn][0] = i0 >= 0 ? ldg64_stream(cnext + jn * cs + i0 * 8 + g) : 0.0;
            bn[jn][1] = i1 >= 0 ? ldg64_stream(cnext + jn * cs + i1 * 8 + g) : 0.0;
        }
        if (GP > 0) {
#pragma unroll
            for (int i = 0; i < GP; i++) {
                dmma(c0, c1, Aw[i][0], bp[i][0]);
                dmma(c0, c1, Aw[i][1], bp[i][1]);
            }
            if (i0 >= 0) st64(R + i0 * 8 + g, c0);
            if (i1 >= 0) st64(R + i1 * 8 + g, c1);
        }
#pragma unroll
        for (int jn = 0; jn < GN; jn++) {
            dmma(D[jn][0], D[jn][1], c0, bn[jn][0]);
            dmma(D[jn][0], D[jn][1], c1, bn[jn][1]);
        }
        rr = fma(c0, c0, fma(c1, c1, rr));
        if (GRAM) {
            int n = 0;
#pragma unroll
            for (int i = 0; i < GN; i++)
#pragma unroll
                for (int jj = i; jj < GN; jj++, n++) {
                    dmma(X[n][0], X[n][1], bn[i][0], bn[jj][0]);
                    dmma(X[n][0], X[n][1], bn[i][1], bn[jj][1]);
                }
        }
    }
    if (GRAM) {
        const int a = g >> 1, ri = g & 1, c = j;
        int n = 0;
#pragma unroll
        for (int i = 0; i < GN; i++)
#pragma unroll
            for (int jj = i; jj < GN; jj++, n++) {
                const double p0 = __shfl_xor_sync(0xffffffffu, X[n][0], 4), p1 = __shfl_xor_sync(0xffffffffu, X[n][1], 4);
                if (ri != 0) continue;
                const double re = X[n][0] + p1, im = p0 - X[n][1];
                if (i == jj) {
                    // packed Hermitian Scc: diagonal [a], then the upper pairs (a < c) in the order of compress.cuh
                    double* o = Scc + ((size_t)(kn0 + i) * B + b) * NSCC_FULL;
                    if (c == a) o[a] = re;
                    else if (a < c) {
                        const int pr = a * 4 - a * (a + 1) / 2 + (c - a - 1);
                        o[4 + 2 * pr] = re;
                        o[5 + 2 * pr] = im;
                    }
                } else {
                    double* o = Xg + ((size_t)grp_pair(i, jj) * B + b) * NX_FULL + 2 * (4 * a + c);
                    o[0] = re;
                    o[1] = im;
                }
            }
    }
    if (GN > 0) {
        const int a = g >> 1, ri = g & 1;
#pragma unroll
        for (int jn = 0; jn < GN; jn++) {
            const double p0 = __shfl_xor_sync(0xffffffffu, D[jn][0], 4), p1 = __shfl_xor_sync(0xffffffffu, D[jn][1], 4);
            if (ri == 0) {
                double* rec = SrcG + ((size_t)jn * B + b) * NSRC_FULL + 2 * (4 * a + j);
                rec[0] = D[jn][0] + p1;
                rec[1] = p0 - D[jn][1];
            }
        }
        for (int o = 16; o > 0; o >>= 1) rr += __shfl_xor_sync(0xffffffffu, rr, o);
        if (lane == 0) {
#pragma unroll
            for (int jn = 0; jn < GN; jn++) {
                double* rec = SrcG + ((size_t)jn * B + b) * NSRC_FULL;
                rec[NSRC_FULL - 2] = rr;
                rec[NSRC_FULL - 1] = 0.0;
            }
        }
    }
}

// Right before cluster j >= 1 of a group is solved: Src_j -= sum_{i<j} dW_i X_ij (the clusters of the group solved so
// far, each Src record read and written once) and srr_j = srr_{j-1} - Re tr(dW_{j-1}^H (Src_{j-1} + Sec_{j-1})), the
// cost per baseline after cluster j-1's update.  4 lanes per baseline, lane a owns row a of dW_i (dP_i[a] in scalar
// form).  J0g / Jg: centre and solved Jones of the group's clusters, [GRP][N][4] each.
template <bool SCALAR>
__global__ void __launch_bounds__(128)
groupfix_kernel(int N, int64_t B, int j, const sagecal_c128* __restrict__ J0g, const sagecal_c128* __restrict__ Jg,
                const double* __restrict__ Scc_prev, const double* __restrict__ Xg, double* __restrict__ SrcG) {
    constexpr int NSRC = SCALAR ? NSRC_SCALAR : NSRC_FULL;
    constexpr int NC = SCALAR ? 1 : 4;
    const int64_t gid = (int64_t)blockIdx.x * 128 + threadIdx.x;
    const int a = (int)(gid & 3);
    const int64_t b = gid >> 2;
    const bool live = b < B;
    const size_t bb = live ? (size_t)b : 0;
    int p, q;
    bl_stations(N, (int64_t)bb, p, q);

    double* sj = SrcG + ((size_t)j * B + bb) * NSRC;
    cplx r[NC];                                          // row a of Src_j (Sr_j[a] in scalar form)
    if (SCALAR) r[0] = mk(sj[2 * a], sj[2 * a + 1]);
    else {
#pragma unroll
        for (int c = 0; c < 4; c++) { const double2 v = reinterpret_cast<const double2*>(sj)[4 * a + c]; r[c] = mk(v.x, v.y); }
    }
    cplx dw[NC];
    for (int i = 0; i < j; i++) {
        const sagecal_c128* J0 = J0g + (size_t)i * N * 4;
        const sagecal_c128* J = Jg + (size_t)i * N * 4;
#pragma unroll
        for (int c = 0; c < NC; c++) dw[c] = SCALAR ? dP_entry(J0, J, p, q, a) : dW_entry(J0, J, p, q, a, c);
        const double* x = Xg + ((size_t)grp_pair(i, j) * B + bb) * (SCALAR ? NX_SCALAR : NX_FULL);
        if (SCALAR) r[0] = cfms(dw[0], mk(x[0], x[1]), r[0]);
        else {
            const double2* x2 = reinterpret_cast<const double2*>(x);      // records are 16-byte aligned
#pragma unroll
            for (int e = 0; e < 4; e++)
#pragma unroll
                for (int c = 0; c < 4; c++) { const double2 v = __ldg(x2 + 4 * e + c); r[c] = cfms(dw[e], mk(v.x, v.y), r[c]); }
        }
    }
    if (live) {
        if (SCALAR) { sj[2 * a] = r[0].re; sj[2 * a + 1] = r[0].im; }
        else {
#pragma unroll
            for (int c = 0; c < 4; c++) reinterpret_cast<double2*>(sj)[4 * a + c] = make_double2(r[c].re, r[c].im);
        }
    }

    // dw now holds row a of dW_{j-1}: srr_j = srr_{j-1} - Re tr(dW^H (Src + Sec)), Sec = Src - dW Scc, of cluster j-1
    const double* si = SrcG + ((size_t)(j - 1) * B + bb) * NSRC;
    double d = 0.0;
    if (SCALAR) {
        const double s2 = Scc_prev[bb];
        const cplx sr = mk(si[2 * a], si[2 * a + 1]);
        const cplx v = mk(2.0 * sr.re - s2 * dw[0].re, 2.0 * sr.im - s2 * dw[0].im);
        d = dw[0].re * v.re + dw[0].im * v.im;
    } else {
        const double* sc = Scc_prev + bb * NSCC_FULL;
#pragma unroll
        for (int c = 0; c < 4; c++) {
            // (dW Scc)[a][c] = sum_e dW[a][e] Scc[e][c], Scc Hermitian from its packed form
            cplx acc = mk(0.0, 0.0);
#pragma unroll
            for (int e = 0; e < 4; e++) {
                cplx sv;
                if (e == c) sv = mk(sc[e], 0.0);
                else {
                    const int lo = e < c ? e : c, hi = e < c ? c : e;
                    const int pr = lo * 4 - lo * (lo + 1) / 2 + (hi - lo - 1);
                    sv = mk(sc[4 + 2 * pr], e < c ? sc[5 + 2 * pr] : -sc[5 + 2 * pr]);
                }
                acc = cfma(dw[e], sv, acc);
            }
            const cplx sr = mk(si[2 * (4 * a + c)], si[2 * (4 * a + c) + 1]);
            const cplx v = mk(2.0 * sr.re - acc.re, 2.0 * sr.im - acc.im);
            d += dw[c].re * v.re + dw[c].im * v.im;      // Re(conj(dW) v)
        }
    }
    d += __shfl_xor_sync(0xffffffffu, d, 1);
    d += __shfl_xor_sync(0xffffffffu, d, 2);
    if (live && a == 0) sj[NSRC - 2] = si[NSRC - 2] - d;
}


// ---- host side ----------------------------------------------------------------------------------------------------
struct WbgArgs {
    int N, T, F;
    sagecal_c128* R;
    const sagecal_c128* coh;
    size_t cstride;
    int kp0, gp;
    const sagecal_c128 *J0prev, *jones;
    int kn0, gn;
    double *SrcG, *Scc, *Xg;
};

template <int GP, int GN>
static void launch_wbgroup_scalar(const WbgArgs& a, cudaStream_t st) {
    const int64_t B = (int64_t)a.N * (a.N - 1) / 2;
    const int FP = stat_group(a.F), BL = WG_THREADS / FP;
    const unsigned grid = (unsigned)((B + BL - 1) / BL);
    if (a.Scc != nullptr && GN > 0)
        wbgroup_scalar_kernel<GP, GN, true><<<grid, WG_THREADS, 0, st>>>(a.N, a.T, a.F, FP, B, a.R, a.coh, a.cstride, a.kp0, a.J0prev, a.jones, a.kn0, a.SrcG, a.Scc, a.Xg);
    else
        wbgroup_scalar_kernel<GP, GN, false><<<grid, WG_THREADS, 0, st>>>(a.N, a.T, a.F, FP, B, a.R, a.coh, a.cstride, a.kp0, a.J0prev, a.jones, a.kn0, a.SrcG, a.Scc, a.Xg);
}
template <int GP, int GN>
static void launch_wbgroup_mma(const WbgArgs& a, cudaStream_t st) {
    const int64_t B = (int64_t)a.N * (a.N - 1) / 2;
    const unsigned grid = (unsigned)((B + MMA_WARPS - 1) / MMA_WARPS);
    const bool gram = a.Scc != nullptr && GN > 0;
#define SGC_WM(F8_, GR_) wbgroup_mma_kernel<GP, GN, F8_, GR_><<<grid, 32 * MMA_WARPS, 0, st>>>(a.N, a.T, a.F, B, a.R, a.coh, a.cstride, a.kp0, a.J0prev, a.jones, a.kn0, a.SrcG, a.Scc, a.Xg)
    if (a.F == 8) { if (gram) SGC_WM(true, true); else SGC_WM(true, false); }
    else { if (gram) SGC_WM(false, true); else SGC_WM(false, false); }
#undef SGC_WM
}
template <bool SCALAR, int GP, int GN>
static void launch_wbgroup_one(const WbgArgs& a, cudaStream_t st) {
    if (GP == 0 && GN == 0) return;
    if (SCALAR) launch_wbgroup_scalar<GP, GN>(a, st);
    else launch_wbgroup_mma<GP, GN>(a, st);
}
template <bool SCALAR, int GP>
static void launch_wbgroup_gn(const WbgArgs& a, cudaStream_t st) {
    switch (a.gn) {
        case 0: launch_wbgroup_one<SCALAR, GP, 0>(a, st); break;
        case 1: launch_wbgroup_one<SCALAR, GP, 1>(a, st); break;
        case 2: launch_wbgroup_one<SCALAR, GP, 2>(a, st); break;
        case 3: launch_wbgroup_one<SCALAR, GP, 3>(a, st); break;
        default: launch_wbgroup_one<SCALAR, GP, 4>(a, st); break;
    }
}
template <bool SCALAR>
static void launch_wbgroup_gp(const WbgArgs& a, cudaStream_t st) {
    switch (a.gp) {
        case 0: launch_wbgroup_gn<SCALAR, 0>(a, st); break;
        case 1: launch_wbgroup_gn<SCALAR, 1>(a, st); break;
        case 2: launch_wbgroup_gn<SCALAR, 2>(a, st); break;
        case 3: launch_wbgroup_gn<SCALAR, 3>(a, st); break;
        default: launch_wbgroup_gn<SCALAR, 4>(a, st); break;
    }
}

int enqueue_wbgroup(int N, int T, int F, int coh_format, sagecal_c128* R, const sagecal_c128* coh, size_t cstride,
                    int kp0, int gp, const sagecal_c128* J0prev, const sagecal_c128* jones, int kn0, int gn,
                    double* SrcG, double* Scc, double* Xgroup, cudaStream_t st) {
    static_assert(GRP == 4, "the dispatch tables above are written for GRP = 4");
    if (gp < 0) gp = 0;
    if (gn < 0) gn = 0;
    if (gp == 0 && gn == 0) return SAGECAL_OK;
    if (gp > GRP || gn > GRP) return SAGECAL_EINVAL;
    const bool scalar = coh_format == SAGECAL_COH_SCALAR;
    const WbgArgs a = {N, T, F, R, coh, cstride, kp0, gp, J0prev, jones, kn0, gn, SrcG, Scc, Xgroup};
    LaunchScope ls(KK_WBSTAT, st);
    if (scalar) launch_wbgroup_gp<true>(a, st);
    else launch_wbgroup_gp<false>(a, st);
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}

int enqueue_groupfix(int N, bool scalar, int j, const sagecal_c128* J0g, const sagecal_c128* Jg, const double* Scc_prev,
                     const double* Xgroup, double* SrcG, cudaStream_t st) {
    if (j < 1 || j >= GRP) return SAGECAL_OK;
    const int64_t B = (int64_t)N * (N - 1) / 2;
    const unsigned grid = (unsigned)((4 * B + 127) / 128);
    LaunchScope ls(KK_GFIX, st);
    if (scalar) groupfix_kernel<true><<<grid, 128, 0, st>>>(N, B, j, J0g, Jg, Scc_prev, Xgroup, SrcG);
    else groupfix_kernel<false><<<grid, 128, 0, st>>>(N, B, j, J0g, Jg, Scc_prev, Xgroup, SrcG);
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}

}  // namespace sgc

using namespace sgc;

// Host-side replay of the tensor-core kernel's fragment addressing (CPU tests, no device needed): for every baseline,
// 8-sample chunk and lane, the doubles the lane touches as C/D/A fragment (and as B fragment of the next group's
// coherencies) -- position lane >> 2 of samples 2 (lane & 3) and 2 (lane & 3) + 1 -- and as B fragment of the previous
// group's coherencies -- positions (lane & 3) and 4 + (lane & 3) of sample lane >> 2.
extern "C" int sagecal_debug_mma_cover(int N, int T, int F, int32_t* cover_cd, int32_t* cover_b) {
    if (N < 2 || T < 1 || F < 1 || !cover_cd || !cover_b) return SAGECAL_EINVAL;
    const int64_t B = (int64_t)N * (N - 1) / 2, nd = (int64_t)T * B * F * 8;
    const int TF = T * F;
    int bad = 0;
    for (int64_t b = 0; b < B; b++)
        for (int m0 = 0; m0 < TF; m0 += 8)
            for (int lane = 0; lane < 32; lane++) {
                const int g = lane >> 2, j = lane & 3;
                const int64_t in = F == 8 ? sample_index<true>(m0 + g, TF, F, B, b) : sample_index<false>(m0 + g, TF, F, B, b);
                const int64_t i0 = F == 8 ? sample_index<true>(m0 + 2 * j, TF, F, B, b) : sample_index<false>(m0 + 2 * j, TF, F, B, b);
                const int64_t i1 = F == 8 ? sample_index<true>(m0 + 2 * j + 1, TF, F, B, b) : sample_index<false>(m0 + 2 * j + 1, TF, F, B, b);
                for (int64_t i : {i0, i1}) {
                    if (i < 0) continue;
                    if (i * 8 + g >= nd) { bad |= 1; continue; }
                    cover_cd[i * 8 + g]++;
                }
                if (in >= 0) {
                    if (in * 8 + 4 + j >= nd) { bad |= 2; continue; }
                    cover_b[in * 8 + j]++;
                    cover_b[in * 8 + 4 + j]++;
                }
            }
    return bad;
}
