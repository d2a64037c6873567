// Cluster-group form of the compressed M-step's streaming kernel (DESIGN.md §5.5 "cluster groups").
//
// wbstat.cu moves 256 B per sample and cluster: R read and written, C_prev, C_next.  The statistics are linear in R,
// so R need not be current when they are taken: for a group of GRP consecutive clusters
//
//   wbgroup:   R <- R - sum_{i in previous group} dW_i c_i          (ONE read and ONE write of R per group)
//              Src_j = sum_tf r c_j^H for every j in the next group, srr = sum_tf |r|^2
//   groupfix:  after cluster i of the group is solved, for the later j of the group
//              Src_j <- Src_j - dW_i X_ij,   X_ij = sum_tf c_i c_j^H   (r' = r - dW_i c_i  =>  r' c_j^H = r c_j^H - dW_i c_i c_j^H)
//              srr_{i+1} = srr_i - Re tr(dW_i^H (Src_i + Sec_i))         (the cost per baseline after i's update)
//   xgram:     X_ij and Scc_i of a group, once per interval (they depend on the coherencies only)
//
// (2 + 2 GRP) x 64 B per sample and group instead of GRP x 256 B: 160 B instead of 256 B per cluster at GRP = 4
// (2x2 coherencies; 64 B instead of 160 B with scalar coherencies).  Nothing is approximated; the LM trajectory is the
// same to rounding.
//
// Thread mapping of the streaming kernels.
//   Scalar coherencies: one thread per (baseline, channel) sample as in wbstat.cu -- 8 accumulators per cluster.
//   2x2 coherencies: 4 lanes share a sample and lane l owns COLUMN l of the 4x4 statistics (r_a conj(c_l), a = 0..3),
//   8 accumulators per cluster instead of 32, so a group fits in registers.  Lane l loads only entry l of every
//   coherency sample and of R (16 B each: a warp reads 512 contiguous bytes per array and time slot, nothing twice --
//   a row-owning layout, where the 4 lanes of a sample each load the whole 64 B, ran at 92 % L1 throughput and 41 %
//   of DRAM throughput).  The write-back needs a product over columns: every lane forms its column's contribution to
//   all four rows and a 2-step reduce-scatter over the quad (12 shuffles) leaves row l in lane l; a 2-step all-gather
//   (12 shuffles) then gives every lane the whole new r for its column of the statistics.
// Sums over the channel lanes of a baseline by warp shuffles, fixed order, no atomics.
#include "compress.cuh"

namespace sgc {

constexpr int WG_THREADS = 128;

// 2x2 coherencies: lanes of one baseline in a warp = 4 (columns) x FP (channels); FP = smallest power of two >= F, <= 8
static inline int group_fp(int F) { int g = 1; while (g < F && g < 8) g <<= 1; return g; }

__device__ __forceinline__ cplx ld_c(const sagecal_c128* p) {     // coherent 16 B load (R is written by this kernel)
    cplx r;
    asm volatile("ld.global.v2.f64 {%0,%1}, [%2];" : "=d"(r.re), "=d"(r.im) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st_c(sagecal_c128* p, cplx v) {
    asm volatile("st.global.v2.f64 [%2], {%0,%1};" ::"d"(v.re), "d"(v.im), "l"(p) : "memory");
}
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ cplx shfl_c(unsigned mask, cplx v, int x) {
    return mk(__shfl_xor_sync(mask, v.re, x), __shfl_xor_sync(mask, v.im, x));
}
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return mk(a.re + b.re, a.im + b.im); }
__device__ __forceinline__ cplx csel(bool s, cplx a, cplx b) { return s ? a : b; }
// sum over lanes l, l ^ stride, l ^ 2 stride, ... (n lanes, n a power of two)
__device__ __forceinline__ double lanes_sum(double v, int n, int stride) {
    for (int o = n >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o * stride);
    return v;
}
// every lane of a quad holds one entry x_l of a 4-vector: afterwards all four lanes hold the whole vector
__device__ __forceinline__ void quad_gather(unsigned qmask, int lane, cplx mine, cplx out[4]) {
    const int qb = lane & ~3;
#pragma unroll
    for (int a = 0; a < 4; a++) out[a] = mk(__shfl_sync(qmask, mine.re, qb + a), __shfl_sync(qmask, mine.im, qb + a));
}
// every lane of a quad holds a 4-vector v: afterwards lane l holds entry l of the sum of the four vectors
__device__ __forceinline__ cplx quad_reduce_scatter(unsigned qmask, int l, const cplx v[4]) {
    const bool odd = l & 1, hi = l & 2;
    const cplx k0 = cadd(csel(hi, v[2], v[0]), shfl_c(qmask, csel(hi, v[0], v[2]), 2));
    const cplx k1 = cadd(csel(hi, v[3], v[1]), shfl_c(qmask, csel(hi, v[1], v[3]), 2));
    return cadd(csel(odd, k1, k0), shfl_c(qmask, csel(odd, k0, k1), 1));
}

// ---- write-back of the previous group + statistics of the next group ------------------------------------------------
template <bool SCALAR, int GP, int GN>
__global__ void __launch_bounds__(WG_THREADS, 3)
wbgroup_kernel(int N, int T, int F, int FP, int64_t B, sagecal_c128* R, const sagecal_c128* __restrict__ coh,
               size_t cstride, int kp0, const sagecal_c128* __restrict__ J0prev, const sagecal_c128* __restrict__ jones,
               int kn0, double* __restrict__ SrcG) {
    constexpr int NW = SCALAR ? 4 : 16;                  // entries of dP / dW per baseline and cluster
    constexpr int LPS = SCALAR ? 1 : 4;                  // lanes per sample
    constexpr int SPC = WG_THREADS / LPS;                // samples per CTA and time slot
    constexpr int NSRC = SCALAR ? NSRC_SCALAR : NSRC_FULL;
    constexpr int GPn = GP > 0 ? GP : 1, GNn = GN > 0 ? GN : 1;
    // scalar: [cluster][entry][baseline] (a warp's lanes differ in the baseline); 2x2: [cluster][baseline][entry], 17
    // entries per row (the 4 lanes of a sample read 4 consecutive entries, baselines fall on different banks)
    constexpr int D1 = SCALAR ? NW : SPC, D2 = SCALAR ? SPC : NW + 1;
    __shared__ cplx s_dw[GPn][D1][D2];
    const int tid = threadIdx.x;
    const int l = SCALAR ? 0 : (tid & 3), s = tid / LPS;
    const int BL = SPC / FP;                             // baselines per CTA
    const int g = s / FP, fl = s - g * FP;
    const int64_t b = (int64_t)blockIdx.x * BL + g;

    if (GP > 0) {
        for (int e = tid; e < BL * NW * GP; e += WG_THREADS) {
            const int i = e / (BL * NW), rem = e - i * (BL * NW);
            const int bl = rem / NW, w = rem - bl * NW;
            const int64_t bb = (int64_t)blockIdx.x * BL + bl;
            cplx v = mk(0.0, 0.0);
            if (bb < B) {
                int p, q;
                bl_stations(N, bb, p, q);
                const sagecal_c128* J0 = J0prev + (size_t)i * N * 4;
                const sagecal_c128* J = jones + (size_t)(kp0 + i) * N * 4;
                v = SCALAR ? dP_entry(J0, J, p, q, w) : dW_entry(J0, J, p, q, w >> 2, w & 3);
            }
            if (SCALAR) s_dw[i][w][bl] = v; else s_dw[i][bl][w] = v;
        }
        __syncthreads();
    }

    cplx S[GNn][4];                                      // scalar: Sr_j[a]; 2x2: column l of Src_j, S[j][a] = Src_j[a][l]
#pragma unroll
    for (int j = 0; j < GNn; j++)
#pragma unroll
        for (int a = 0; a < 4; a++) S[j][a] = mk(0.0, 0.0);
    double rr = 0.0;

    if (b < B) {
        const sagecal_c128* cprev = coh + (size_t)kp0 * cstride;
        const sagecal_c128* cnext = coh + (size_t)kn0 * cstride;
        const size_t step = (size_t)B * F;
        const unsigned qmask = SCALAR ? 0u : (0xFu << ((tid & 31) & ~3));
        for (int f = fl; f < F; f += FP) {
            size_t idx = (size_t)b * F + f;
#pragma unroll 1
            for (int t = 0; t < T; t++, idx += step) {
                cplx cp[GPn], cn[GNn];
                if (SCALAR) {
                    m22 r;
                    load_m22(R + idx * 4, r);
#pragma unroll
                    for (int i = 0; i < GP; i++) cp[i] = ldg128_stream(cprev + (size_t)i * cstride + idx);
#pragma unroll
                    for (int j = 0; j < GN; j++) cn[j] = ldg128_stream(cnext + (size_t)j * cstride + idx);
#pragma unroll
                    for (int i = 0; i < GP; i++)
#pragma unroll
                        for (int a = 0; a < 4; a++) r.a[a] = cfms(s_dw[i][a][g], cp[i], r.a[a]);
                    if (GP > 0) store_m22(R + idx * 4, r);
#pragma unroll
                    for (int j = 0; j < GN; j++)
#pragma unroll
                        for (int a = 0; a < 4; a++) S[j][a] = cfmac(r.a[a], cn[j], S[j][a]);
                    rr = cabs2(r.a[3], cabs2(r.a[2], cabs2(r.a[1], cabs2(r.a[0], rr))));
                } else {
                    cplx rl = ld_c(R + idx * 4 + l);                     // r_l
#pragma unroll
                    for (int i = 0; i < GP; i++) cp[i] = ldg128_stream(cprev + (size_t)i * cstride + idx * 4 + l);
#pragma unroll
                    for (int j = 0; j < GN; j++) cn[j] = ldg128_stream(cnext + (size_t)j * cstride + idx * 4 + l);
                    if (GP > 0) {
                        // column l of the write-back: v[a] = sum_i dW_i[a][l] c_i[l]; row l of the total to lane l
                        cplx v[4];
#pragma unroll
                        for (int a = 0; a < 4; a++) v[a] = mk(0.0, 0.0);
#pragma unroll
                        for (int i = 0; i < GP; i++)
#pragma unroll
                            for (int a = 0; a < 4; a++) v[a] = cfma(s_dw[i][g][4 * a + l], cp[i], v[a]);
                        const cplx w = quad_reduce_scatter(qmask, l, v);
                        rl = mk(rl.re - w.re, rl.im - w.im);
                        st_c(R + idx * 4 + l, rl);
                    }
                    if (GN > 0) {
                        cplx r[4];
                        quad_gather(qmask, tid & 31, rl, r);
#pragma unroll
                        for (int j = 0; j < GN; j++)
#pragma unroll
                            for (int a = 0; a < 4; a++) S[j][a] = cfmac(r[a], cn[j], S[j][a]);
                    }
                    rr = cabs2(rl, rr);
                }
            }
        }
    }
    if (GN > 0) {
        const bool writer = fl == 0 && b < B;
        const size_t bb = b < B ? (size_t)b : 0;
#pragma unroll
        for (int j = 0; j < GN; j++) {
            double* rec = SrcG + ((size_t)j * B + bb) * NSRC;
#pragma unroll
            for (int a = 0; a < 4; a++) {
                const double re = lanes_sum(S[j][a].re, FP, LPS), im = lanes_sum(S[j][a].im, FP, LPS);
                if (writer) {
                    const int e = SCALAR ? a : 4 * a + l;
                    rec[2 * e] = re;
                    rec[2 * e + 1] = im;
                }
            }
        }
        rr = lanes_sum(rr, FP * LPS, 1);
        if (writer && l == 0) {
#pragma unroll
            for (int j = 0; j < GN; j++) {
                double* rec = SrcG + ((size_t)j * B + bb) * NSRC;
                rec[NSRC - 2] = rr;        // meaningful for j = 0; groupfix rewrites it for the later clusters
                rec[NSRC - 1] = 0.0;
            }
        }
    }
}

// ---- Scc_i and X_ij (i < j) of the GN clusters kn0.. of a group -------------------------------------------------------
// 2x2: lane l owns column l, X_ij[a][l] = sum c_i[a] conj(c_j[l]); the rows c_i[a] come from the quad by an all-gather.
template <bool SCALAR, int GN>
__global__ void __launch_bounds__(WG_THREADS, SCALAR ? 4 : 2)
xgram_kernel(int T, int F, int FP, int64_t B, const sagecal_c128* __restrict__ coh, size_t cstride, int kn0,
             double* __restrict__ Scc, double* __restrict__ Xg) {
    constexpr int NR = SCALAR ? 1 : 4;
    constexpr int LPS = SCALAR ? 1 : 4;
    constexpr int SPC = WG_THREADS / LPS;
    constexpr int NP = GN * (GN + 1) / 2;                // pairs i <= j
    const int tid = threadIdx.x;
    const int l = SCALAR ? 0 : (tid & 3), s = tid / LPS;
    const int BL = SPC / FP;
    const int g = s / FP, fl = s - g * FP;
    const int64_t b = (int64_t)blockIdx.x * BL + g;
    cplx X[NP][NR];
#pragma unroll
    for (int n = 0; n < NP; n++)
#pragma unroll
        for (int a = 0; a < NR; a++) X[n][a] = mk(0.0, 0.0);

    if (b < B) {
        const sagecal_c128* cb = coh + (size_t)kn0 * cstride;
        const size_t step = (size_t)B * F;
        const unsigned qmask = SCALAR ? 0u : (0xFu << ((tid & 31) & ~3));
        for (int f = fl; f < F; f += FP) {
            size_t idx = (size_t)b * F + f;
#pragma unroll 1
            for (int t = 0; t < T; t++, idx += step) {
                cplx c[GN];
#pragma unroll
                for (int i = 0; i < GN; i++) c[i] = ldg128_stream(cb + (size_t)i * cstride + idx * LPS + l);
                if (!SCALAR && t + 2 < T && l < GN) prefetch_l2(cb + (size_t)l * cstride + (idx + 2 * step) * 4);
                int n = 0;
#pragma unroll
                for (int i = 0; i < GN; i++) {
                    cplx ci[4];
                    if (SCALAR) ci[0] = c[i];
                    else quad_gather(qmask, tid & 31, c[i], ci);
#pragma unroll
                    for (int j = i; j < GN; j++, n++)
#pragma unroll
                        for (int a = 0; a < NR; a++) X[n][a] = cfmac(ci[a], c[j], X[n][a]);
                }
            }
        }
    }
    const bool writer = fl == 0 && b < B;
    const size_t bb = b < B ? (size_t)b : 0;
    int n = 0;
#pragma unroll
    for (int i = 0; i < GN; i++) {
#pragma unroll
        for (int j = i; j < GN; j++, n++) {
            double re[NR], im[NR];
#pragma unroll
            for (int a = 0; a < NR; a++) { re[a] = lanes_sum(X[n][a].re, FP, LPS); im[a] = lanes_sum(X[n][a].im, FP, LPS); }
            if (!writer) continue;
            if (i == j) {
                double* o = Scc + ((size_t)(kn0 + i) * B + bb) * (SCALAR ? NSCC_SCALAR : NSCC_FULL);
                if (SCALAR) o[0] = re[0];
                else {
                    // packed Hermitian: diagonal [l], then the upper pairs (a < l, l) in the order of compress.cuh
#pragma unroll
                    for (int a = 0; a < NR; a++) {
                        if (a == l) o[l] = re[a];
                        else if (a < l) {
                            const int pr = a * 4 - a * (a + 1) / 2 + (l - a - 1);
                            o[4 + 2 * pr] = re[a];
                            o[5 + 2 * pr] = im[a];
                        }
                    }
                }
            } else {
                double* o = Xg + ((size_t)grp_pair(i, j) * B + bb) * (SCALAR ? NX_SCALAR : NX_FULL);
                if (SCALAR) { o[0] = re[0]; o[1] = im[0]; }
                else {
#pragma unroll
                    for (int a = 0; a < NR; a++) { o[2 * (4 * a + l)] = re[a]; o[2 * (4 * a + l) + 1] = im[a]; }
                }
            }
        }
    }
}

// 4 lanes per baseline, lane a owns row a of dW_i (dP_i[a] in scalar form).
template <bool SCALAR>
__global__ void __launch_bounds__(128)
groupfix_kernel(int N, int64_t B, int i, int gn, const sagecal_c128* __restrict__ J0, const sagecal_c128* __restrict__ J,
                const double* __restrict__ Scc_i, const double* __restrict__ Xg, double* __restrict__ SrcG) {
    constexpr int NSRC = SCALAR ? NSRC_SCALAR : NSRC_FULL;
    constexpr int NC = SCALAR ? 1 : 4;
    const int64_t gid = (int64_t)blockIdx.x * 128 + threadIdx.x;
    const int a = (int)(gid & 3);
    const int64_t b = gid >> 2;
    const bool live = b < B;
    const size_t bb = live ? (size_t)b : 0;
    int p, q;
    bl_stations(N, (int64_t)bb, p, q);
    cplx dw[NC];
#pragma unroll
    for (int c = 0; c < NC; c++) dw[c] = SCALAR ? dP_entry(J0, J, p, q, a) : dW_entry(J0, J, p, q, a, c);

    // srr after cluster i's update: srr - Re tr(dW^H (Src_i + Sec_i)), Sec_i = Src_i - dW Scc_i
    const double* si = SrcG + ((size_t)i * B + bb) * NSRC;
    double d = 0.0;
    if (SCALAR) {
        const double s2 = Scc_i[bb];
        const cplx sr = mk(si[2 * a], si[2 * a + 1]);
        const cplx v = mk(2.0 * sr.re - s2 * dw[0].re, 2.0 * sr.im - s2 * dw[0].im);
        d = dw[0].re * v.re + dw[0].im * v.im;
    } else {
        const double* sc = Scc_i + bb * NSCC_FULL;
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
    if (live && a == 0 && i + 1 < gn) SrcG[((size_t)(i + 1) * B + bb) * NSRC + NSRC - 2] = si[NSRC - 2] - d;

    // Src_j -= dW_i X_ij for the later clusters of the group
    for (int j = i + 1; j < gn; j++) {
        const double* x = Xg + ((size_t)grp_pair(i, j) * B + bb) * (SCALAR ? NX_SCALAR : NX_FULL);
        double* sj = SrcG + ((size_t)j * B + bb) * NSRC;
        if (SCALAR) {
            const cplx r = cfms(dw[0], mk(x[0], x[1]), mk(sj[2 * a], sj[2 * a + 1]));
            if (live) { sj[2 * a] = r.re; sj[2 * a + 1] = r.im; }
        } else {
#pragma unroll
            for (int c = 0; c < 4; c++) {
                cplx r = mk(sj[2 * (4 * a + c)], sj[2 * (4 * a + c) + 1]);
#pragma unroll
                for (int e = 0; e < 4; e++) r = cfms(dw[e], mk(x[2 * (4 * e + c)], x[2 * (4 * e + c) + 1]), r);
                if (live) { sj[2 * (4 * a + c)] = r.re; sj[2 * (4 * a + c) + 1] = r.im; }
            }
        }
    }
}


// ---- host side ----------------------------------------------------------------------------------------------------
template <bool SCALAR, int GP>
static void launch_wbgroup_gn(int gn, unsigned grid, cudaStream_t st, int N, int T, int F, int FP, int64_t B,
                              sagecal_c128* R, const sagecal_c128* coh, size_t cstride, int kp0,
                              const sagecal_c128* J0prev, const sagecal_c128* jones, int kn0, double* SrcG) {
#define SGC_WG(GN_) wbgroup_kernel<SCALAR, GP, GN_><<<grid, WG_THREADS, 0, st>>>(N, T, F, FP, B, R, coh, cstride, kp0, J0prev, jones, kn0, SrcG)
    switch (gn) {
        case 0: if (GP > 0) SGC_WG(0); break;
        case 1: SGC_WG(1); break;
        case 2: SGC_WG(2); break;
        case 3: SGC_WG(3); break;
        default: SGC_WG(4); break;
    }
#undef SGC_WG
}

template <bool SCALAR>
static int launch_wbgroup(int N, int T, int F, sagecal_c128* R, const sagecal_c128* coh, size_t cstride, int kp0, int gp,
                          const sagecal_c128* J0prev, const sagecal_c128* jones, int kn0, int gn, double* SrcG,
                          cudaStream_t st) {
    const int64_t B = (int64_t)N * (N - 1) / 2;
    const int FP = SCALAR ? stat_group(F) : group_fp(F), BL = (SCALAR ? WG_THREADS : WG_THREADS / 4) / FP;
    const unsigned grid = (unsigned)((B + BL - 1) / BL);
    LaunchScope ls(KK_WBSTAT, st);
#define SGC_GP(GP_) launch_wbgroup_gn<SCALAR, GP_>(gn, grid, st, N, T, F, FP, B, R, coh, cstride, kp0, J0prev, jones, kn0, SrcG)
    switch (gp) {
        case 0: SGC_GP(0); break;
        case 1: SGC_GP(1); break;
        case 2: SGC_GP(2); break;
        case 3: SGC_GP(3); break;
        default: SGC_GP(4); break;
    }
#undef SGC_GP
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}

int enqueue_wbgroup(int N, int T, int F, int coh_format, sagecal_c128* R, const sagecal_c128* coh, size_t cstride,
                    int kp0, int gp, const sagecal_c128* J0prev, const sagecal_c128* jones, int kn0, int gn,
                    double* SrcG, cudaStream_t st) {
    static_assert(GRP == 4, "the dispatch tables above are written for GRP = 4");
    if (gp <= 0 && gn <= 0) return SAGECAL_OK;
    if (gp > GRP || gn > GRP) return SAGECAL_EINVAL;
    return coh_format == SAGECAL_COH_SCALAR
               ? launch_wbgroup<true>(N, T, F, R, coh, cstride, kp0, gp < 0 ? 0 : gp, J0prev, jones, kn0, gn < 0 ? 0 : gn, SrcG, st)
               : launch_wbgroup<false>(N, T, F, R, coh, cstride, kp0, gp < 0 ? 0 : gp, J0prev, jones, kn0, gn < 0 ? 0 : gn, SrcG, st);
}

template <bool SCALAR>
static int launch_xgram(int N, int T, int F, const sagecal_c128* coh, size_t cstride, int kn0, int gn, double* Scc,
                        double* Xg, cudaStream_t st) {
    const int64_t B = (int64_t)N * (N - 1) / 2;
    const int FP = SCALAR ? stat_group(F) : group_fp(F), BL = (SCALAR ? WG_THREADS : WG_THREADS / 4) / FP;
    const unsigned grid = (unsigned)((B + BL - 1) / BL);
    LaunchScope ls(KK_XGRAM, st);
#define SGC_XG(GN_) xgram_kernel<SCALAR, GN_><<<grid, WG_THREADS, 0, st>>>(T, F, FP, B, coh, cstride, kn0, Scc, Xg)
    switch (gn) {
        case 1: SGC_XG(1); break;
        case 2: SGC_XG(2); break;
        case 3: SGC_XG(3); break;
        default: SGC_XG(4); break;
    }
#undef SGC_XG
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}

int enqueue_xgram(int N, int T, int F, int coh_format, const sagecal_c128* coh, size_t cstride, int kn0, int gn,
                  double* Scc, double* Xgroup, cudaStream_t st) {
    if (gn < 1 || gn > GRP) return SAGECAL_EINVAL;
    return coh_format == SAGECAL_COH_SCALAR ? launch_xgram<true>(N, T, F, coh, cstride, kn0, gn, Scc, Xgroup, st)
                                            : launch_xgram<false>(N, T, F, coh, cstride, kn0, gn, Scc, Xgroup, st);
}

int enqueue_groupfix(int N, bool scalar, int i, int gn, const sagecal_c128* J0_i, const sagecal_c128* J_i,
                     const double* Scc_i, const double* Xgroup, double* SrcG, cudaStream_t st) {
    if (i + 1 >= gn) return SAGECAL_OK;
    const int64_t B = (int64_t)N * (N - 1) / 2;
    const unsigned grid = (unsigned)((4 * B + 127) / 128);
    LaunchScope ls(KK_GFIX, st);
    if (scalar) groupfix_kernel<true><<<grid, 128, 0, st>>>(N, B, i, gn, J0_i, J_i, Scc_i, Xgroup, SrcG);
    else groupfix_kernel<false><<<grid, 128, 0, st>>>(N, B, i, gn, J0_i, J_i, Scc_i, Xgroup, SrcG);
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}

}  // namespace sgc
