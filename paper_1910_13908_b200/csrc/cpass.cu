// Compressed LM evaluation pass: cost, gradient and per-station J^H J of one cluster at a trial Jones, from the
// per-baseline statistics of wbstat.cu instead of the T*F samples (formulas and layout: compress.cuh).
// The statistics of one cluster (392 B per baseline, 51 MB at N=512) stay L2-resident over the n_lm+1 evaluations.
//
// Tiling: CTA = (block of 16 row stations p) x (tile of 32 column stations q), lane <-> q, the 4 warps walk the rows.
// Row-station sums are reduced across the lanes with shuffles (one record per tile and row), column-station sums
// stay in registers over the rows and are combined across the warps through shared memory (one record per tile and
// column); creduce_kernel adds each station's records in a fixed order.  No atomics; bit-reproducible.
#include "compress.cuh"

namespace sgc {

struct CSide {
    cplx G[4];
    double M00, M11;
    cplx M01;
    __device__ __forceinline__ void zero() {
        G[0] = G[1] = G[2] = G[3] = M01 = mk(0.0, 0.0);
        M00 = M11 = 0.0;
    }
    __device__ __forceinline__ double get(int i) const {
        switch (i) {
            case 0: return G[0].re; case 1: return G[0].im; case 2: return G[1].re; case 3: return G[1].im;
            case 4: return G[2].re; case 5: return G[2].im; case 6: return G[3].re; case 7: return G[3].im;
            case 8: return M00; case 9: return M11; case 10: return M01.re; default: return M01.im;
        }
    }
};

__device__ __forceinline__ double warp_sum32(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ cplx cconj(cplx a) { return mk(a.re, -a.im); }
__device__ __forceinline__ void gram22(const m22& J, double& h00, double& h11, cplx& h01) {  // H = J^H J
    h00 = cabs2(J.a[2], cabs2(J.a[0], 0.0));
    h11 = cabs2(J.a[3], cabs2(J.a[1], 0.0));
    h01 = cfmaca(J.a[2], J.a[3], cfmaca(J.a[0], J.a[1], mk(0.0, 0.0)));
}
__device__ __forceinline__ void msub(const m22& a, const m22& b, m22& o) {
#pragma unroll
    for (int i = 0; i < 4; i++) o.a[i] = mk(a.a[i].re - b.a[i].re, a.a[i].im - b.a[i].im);
}

// one baseline, general 2x2 coherencies
__device__ __forceinline__ void baseline_full(const double* __restrict__ Src, const double* __restrict__ srr,
                                              const double* __restrict__ Scc, int64_t B, int64_t b, const m22& Jp,
                                              const m22& Dp, const m22& Jq, const m22& Jq0, const m22& Dq, double hp00,
                                              double hp11, cplx hp01, double hq00, double hq11, cplx hq01, CSide& sp,
                                              CSide& sq, double& cost) {
    // Hermitian Scc as a full 4x4
    cplx S[4][4];
#pragma unroll
    for (int a = 0; a < 4; a++) S[a][a] = mk(__ldg(Scc + (size_t)a * B + b), 0.0);
    {
        int pr = 0;
#pragma unroll
        for (int a = 0; a < 4; a++) {
#pragma unroll
            for (int c = a + 1; c < 4; c++, pr++) {
                S[a][c] = mk(__ldg(Scc + (size_t)(4 + 2 * pr) * B + b), __ldg(Scc + (size_t)(5 + 2 * pr) * B + b));
                S[c][a] = cconj(S[a][c]);
            }
        }
    }
    double acc = 0.0;
#pragma unroll
    for (int a = 0; a < 4; a++) {
        const int i = a >> 1, j = a & 1;
        cplx dW[4], src[4], sec[4];
#pragma unroll
        for (int c = 0; c < 4; c++) {
            const int k = c >> 1, l = c & 1;
            dW[c] = cfmac(Jp.a[2 * i + k], Dq.a[2 * j + l], cmulc(Dp.a[2 * i + k], Jq0.a[2 * j + l]));
            src[c] = mk(__ldg(Src + (size_t)(2 * (4 * a + c)) * B + b), __ldg(Src + (size_t)(2 * (4 * a + c) + 1) * B + b));
        }
#pragma unroll
        for (int c = 0; c < 4; c++) {
            cplx s = src[c];
#pragma unroll
            for (int d = 0; d < 4; d++) s = cfms(dW[d], S[d][c], s);
            sec[c] = s;
            // Re(conj(dW) (src + sec))
            const double tr = src[c].re + s.re, ti = src[c].im + s.im;
            acc = fma(dW[c].re, tr, fma(dW[c].im, ti, acc));
        }
        // G_p[i,k] += sum_l J_q[j,l] sec[(k,l)]
#pragma unroll
        for (int k = 0; k < 2; k++)
            sp.G[2 * i + k] = cfma(Jq.a[2 * j + 1], sec[2 * k + 1], cfma(Jq.a[2 * j], sec[2 * k], sp.G[2 * i + k]));
        // G_q[j,l] += sum_k J_p[i,k] conj(sec[(k,l)])
#pragma unroll
        for (int l = 0; l < 2; l++)
            sq.G[2 * j + l] = cfmac(Jp.a[2 * i + 1], sec[2 + l], cfmac(Jp.a[2 * i], sec[l], sq.G[2 * j + l]));
    }
    cost += __ldg(srr + b) - acc;
    // M_p[k,k'] = sum_{l,l'} Hq[l,l'] S[(k,l)][(k',l')]
    sp.M00 += fma(hq00, S[0][0].re, fma(hq11, S[1][1].re, 2.0 * fma(hq01.re, S[0][1].re, -hq01.im * S[0][1].im)));
    sp.M11 += fma(hq00, S[2][2].re, fma(hq11, S[3][3].re, 2.0 * fma(hq01.re, S[2][3].re, -hq01.im * S[2][3].im)));
    {
        cplx m = mk(hq00 * S[0][2].re, hq00 * S[0][2].im);
        m = cfma(hq01, S[0][3], m);
        m = cfma(cconj(hq01), S[1][2], m);
        m = mk(fma(hq11, S[1][3].re, m.re), fma(hq11, S[1][3].im, m.im));
        sp.M01 = mk(sp.M01.re + m.re, sp.M01.im + m.im);
    }
    // M_q[l,l'] = sum_{k,k'} Hp[k,k'] conj(S[(k,l)][(k',l')])
    sq.M00 += fma(hp00, S[0][0].re, fma(hp11, S[2][2].re, 2.0 * fma(hp01.re, S[0][2].re, hp01.im * S[0][2].im)));
    sq.M11 += fma(hp00, S[1][1].re, fma(hp11, S[3][3].re, 2.0 * fma(hp01.re, S[1][3].re, hp01.im * S[1][3].im)));
    {
        cplx m = mk(hp00 * S[0][1].re, -hp00 * S[0][1].im);      // Hp00 conj(S[0][1])
        m = cfmac(hp01, S[0][3], m);                              // Hp01 conj(S[0][3])
        m = cfma(cconj(hp01), S[1][2], m);                        // Hp10 conj(S[2][1]) = conj(Hp01) S[1][2]
        m = mk(fma(hp11, S[2][3].re, m.re), fma(-hp11, S[2][3].im, m.im));   // Hp11 conj(S[2][3])
        sq.M01 = mk(sq.M01.re + m.re, sq.M01.im + m.im);
    }
}

// one baseline, scalar coherencies
__device__ __forceinline__ void baseline_scalar(const double* __restrict__ Src, const double* __restrict__ srr,
                                                const double* __restrict__ Scc, int64_t B, int64_t b, const m22& Jp,
                                                const m22& Dp, const m22& Jq, const m22& Jq0, const m22& Dq,
                                                double hp00, double hp11, cplx hp01, double hq00, double hq11,
                                                cplx hq01, CSide& sp, CSide& sq, double& cost) {
    const double s2 = __ldg(Scc + b);
    m22 dP, t, Se;
    mmh(Dp, Jq0, dP);           // D_p J0_q^H
    mmh(Jp, Dq, t);             // J_p D_q^H
    double acc = 0.0;
#pragma unroll
    for (int a = 0; a < 4; a++) {
        dP.a[a] = mk(dP.a[a].re + t.a[a].re, dP.a[a].im + t.a[a].im);
        const cplx sr = mk(__ldg(Src + (size_t)(2 * a) * B + b), __ldg(Src + (size_t)(2 * a + 1) * B + b));
        Se.a[a] = mk(fma(-s2, dP.a[a].re, sr.re), fma(-s2, dP.a[a].im, sr.im));
        acc = fma(dP.a[a].re, sr.re + Se.a[a].re, fma(dP.a[a].im, sr.im + Se.a[a].im, acc));
    }
    cost += __ldg(srr + b) - acc;
    // G_p += Se J_q;  G_q += Se^H J_p
    sp.G[0] = cfma(Se.a[1], Jq.a[2], cfma(Se.a[0], Jq.a[0], sp.G[0]));
    sp.G[1] = cfma(Se.a[1], Jq.a[3], cfma(Se.a[0], Jq.a[1], sp.G[1]));
    sp.G[2] = cfma(Se.a[3], Jq.a[2], cfma(Se.a[2], Jq.a[0], sp.G[2]));
    sp.G[3] = cfma(Se.a[3], Jq.a[3], cfma(Se.a[2], Jq.a[1], sp.G[3]));
    sq.G[0] = cfmaca(Se.a[2], Jp.a[2], cfmaca(Se.a[0], Jp.a[0], sq.G[0]));
    sq.G[1] = cfmaca(Se.a[2], Jp.a[3], cfmaca(Se.a[0], Jp.a[1], sq.G[1]));
    sq.G[2] = cfmaca(Se.a[3], Jp.a[2], cfmaca(Se.a[1], Jp.a[0], sq.G[2]));
    sq.G[3] = cfmaca(Se.a[3], Jp.a[3], cfmaca(Se.a[1], Jp.a[1], sq.G[3]));
    sp.M00 = fma(s2, hq00, sp.M00); sp.M11 = fma(s2, hq11, sp.M11);
    sp.M01 = mk(fma(s2, hq01.re, sp.M01.re), fma(s2, hq01.im, sp.M01.im));
    sq.M00 = fma(s2, hp00, sq.M00); sq.M11 = fma(s2, hp11, sq.M11);
    sq.M01 = mk(fma(s2, hp01.re, sq.M01.re), fma(s2, hp01.im, sq.M01.im));
}

template <bool SCALAR>
__global__ void __launch_bounds__(CP_THREADS)
cpass_kernel(int N, int64_t B, const double* __restrict__ Src, const double* __restrict__ srr,
             const double* __restrict__ Scc, const sagecal_c128* __restrict__ J0, const sagecal_c128* __restrict__ Jt,
             double* __restrict__ Ppart, double* __restrict__ Qpart) {
    __shared__ double s_q[CP_THREADS / 32][CP_NQ][32];
    const int pb = blockIdx.x, qt = blockIdx.y;
    const int q0 = CP_TQ * qt, qmax = min(N, q0 + CP_TQ) - 1;   // largest q of the tile
    const int p0 = CP_PB * pb;
    if (p0 >= qmax) return;                                     // tile below the diagonal: creduce never reads it
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int q = q0 + lane;
    m22 Jq, Jq0, Dq;
    load_jones(Jt + (size_t)min(q, N - 1) * 4, Jq);
    load_jones(J0 + (size_t)min(q, N - 1) * 4, Jq0);
    msub(Jq, Jq0, Dq);
    double hq00, hq11;
    cplx hq01;
    gram22(Jq, hq00, hq11, hq01);
    CSide sq;
    sq.zero();
    for (int r = warp; r < CP_PB; r += CP_THREADS / 32) {
        const int p = p0 + r;
        if (p >= N - 1) break;                                  // warp-uniform
        m22 Jp, Jp0, Dp;
        load_jones(Jt + (size_t)p * 4, Jp);
        load_jones(J0 + (size_t)p * 4, Jp0);
        msub(Jp, Jp0, Dp);
        double hp00, hp11;
        cplx hp01;
        gram22(Jp, hp00, hp11, hp01);
        CSide sp;
        sp.zero();
        double cost = 0.0;
        if (q > p && q < N) {
            const int64_t b = bl_index(N, p, q);
            if (SCALAR) baseline_scalar(Src, srr, Scc, B, b, Jp, Dp, Jq, Jq0, Dq, hp00, hp11, hp01, hq00, hq11, hq01, sp, sq, cost);
            else baseline_full(Src, srr, Scc, B, b, Jp, Dp, Jq, Jq0, Dq, hp00, hp11, hp01, hq00, hq11, hq01, sp, sq, cost);
        }
        double* out = Ppart + ((size_t)qt * N + p) * CP_NP;
#pragma unroll
        for (int i = 0; i < CP_NQ; i++) {
            const double s = warp_sum32(sp.get(i));
            if (lane == 0) out[i] = s;
        }
        const double cs = warp_sum32(cost);
        if (lane == 0) out[CP_NQ] = cs;
    }
#pragma unroll
    for (int i = 0; i < CP_NQ; i++) s_q[warp][i][lane] = sq.get(i);
    __syncthreads();
    for (int o = threadIdx.x; o < CP_NQ * 32; o += CP_THREADS) {
        const int i = o >> 5, l = o & 31;
        if (q0 + l < N) {
            double s = s_q[0][i][l];
#pragma unroll
            for (int w = 1; w < CP_THREADS / 32; w++) s += s_q[w][i][l];
            Qpart[((size_t)pb * N + q0 + l) * CP_NQ + i] = s;
        }
    }
}

// one warp per station: adds the station's row-side records (tiles qt >= (s+1)/32) and column-side records
// (blocks pb with 16 pb < qmax(s/32)), lanes over records, then a butterfly: fixed order.
constexpr int CR_THREADS = 128;
__global__ void __launch_bounds__(CR_THREADS)
creduce_kernel(CGeom g, const double* __restrict__ Ppart, const double* __restrict__ Qpart,
               double* __restrict__ cost_st, sagecal_c128* __restrict__ grad, sagecal_c128* __restrict__ jtj) {
    const int lane = threadIdx.x & 31;
    const int s = blockIdx.x * (CR_THREADS / 32) + (threadIdx.x >> 5);
    if (s >= g.N) return;
    const int N = g.N;
    double acc[CP_NP];
#pragma unroll
    for (int i = 0; i < CP_NP; i++) acc[i] = 0.0;
    if (s <= N - 2) {
        for (int qt = (s + 1) / CP_TQ + lane; qt < g.nqt; qt += 32) {
            const double* rec = Ppart + ((size_t)qt * N + s) * CP_NP;
#pragma unroll
            for (int i = 0; i < CP_NP; i++) acc[i] += rec[i];
        }
    }
    if (s >= 1) {
        const int qmax = min(N, CP_TQ * (s / CP_TQ) + CP_TQ) - 1;
        const int npb = min(g.npb, (qmax - 1) / CP_PB + 1);
        for (int pb = lane; pb < npb; pb += 32) {
            const double* rec = Qpart + ((size_t)pb * N + s) * CP_NQ;
#pragma unroll
            for (int i = 0; i < CP_NQ; i++) acc[i] += rec[i];
        }
    }
#pragma unroll
    for (int i = 0; i < CP_NP; i++) acc[i] = warp_sum32(acc[i]);
    if (lane == 0) {
        sagecal_c128* G = grad + (size_t)s * 4;
        sagecal_c128* M = jtj + (size_t)s * 4;
        for (int i = 0; i < 4; i++) { G[i].re = acc[2 * i]; G[i].im = acc[2 * i + 1]; }
        M[0].re = acc[8];  M[0].im = 0.0;
        M[1].re = acc[10]; M[1].im = acc[11];
        M[2].re = acc[10]; M[2].im = -acc[11];
        M[3].re = acc[9];  M[3].im = 0.0;
        cost_st[s] = acc[12];
    }
}

size_t compress_workspace_bytes(int N, int K, bool scalar) {
    const CGeom g = make_cgeom(N);
    size_t n = 0;
    n += round_up(sizeof(double) * (size_t)(K > 0 ? K : 1) * nscc(scalar) * g.B, 256);
    n += round_up(sizeof(double) * (size_t)nsrc(scalar) * g.B, 256);
    n += round_up(sizeof(double) * (size_t)g.B, 256);
    n += round_up(sizeof(double) * (size_t)g.nqt * N * CP_NP, 256);
    n += round_up(sizeof(double) * (size_t)g.npb * N * CP_NQ, 256);
    n += round_up(sizeof(double) * (size_t)N, 256);
    n += round_up((size_t)2 * N * 64, 256);
    return n;
}

CompressWorkspace carve_compress(int N, int K, bool scalar, void* ws) {
    const CGeom g = make_cgeom(N);
    CompressWorkspace w;
    char* p = (char*)ws;
    w.Scc = (double*)p; p += round_up(sizeof(double) * (size_t)(K > 0 ? K : 1) * nscc(scalar) * g.B, 256);
    w.Src = (double*)p; p += round_up(sizeof(double) * (size_t)nsrc(scalar) * g.B, 256);
    w.srr = (double*)p; p += round_up(sizeof(double) * (size_t)g.B, 256);
    w.Ppart = (double*)p; p += round_up(sizeof(double) * (size_t)g.nqt * N * CP_NP, 256);
    w.Qpart = (double*)p; p += round_up(sizeof(double) * (size_t)g.npb * N * CP_NQ, 256);
    w.cost_st = (double*)p; p += round_up(sizeof(double) * (size_t)N, 256);
    w.J0 = (sagecal_c128*)p;
    return w;
}

int enqueue_cpass(const CGeom& g, const CompressWorkspace& w, bool scalar, const double* Scc_k, const sagecal_c128* J0,
                  const sagecal_c128* Jt, sagecal_c128* grad, sagecal_c128* jtj, cudaStream_t st) {
    {
        LaunchScope ls(KK_CPASS, st);
        const dim3 grid((unsigned)g.npb, (unsigned)g.nqt);
        if (scalar) cpass_kernel<true><<<grid, CP_THREADS, 0, st>>>(g.N, g.B, w.Src, w.srr, Scc_k, J0, Jt, w.Ppart, w.Qpart);
        else cpass_kernel<false><<<grid, CP_THREADS, 0, st>>>(g.N, g.B, w.Src, w.srr, Scc_k, J0, Jt, w.Ppart, w.Qpart);
        SGC_LAUNCH_CHECK();
    }
    {
        LaunchScope ls(KK_CREDUCE, st);
        const unsigned grid = (unsigned)((g.N + CR_THREADS / 32 - 1) / (CR_THREADS / 32));
        creduce_kernel<<<grid, CR_THREADS, 0, st>>>(g, w.Ppart, w.Qpart, w.cost_st, grad, jtj);
        SGC_LAUNCH_CHECK();
    }
    return SAGECAL_OK;
}

}  // namespace sgc

using namespace sgc;

// Host-side replay of cpass_kernel's tiling and creduce_kernel's record lists (CPU tests, no device needed).
extern "C" int sagecal_debug_cpass_cover(int N, int32_t* cover, int64_t* info) {
    if (N < 2 || !cover || !info) return SAGECAL_EINVAL;
    const CGeom g = make_cgeom(N);
    const size_t nP = (size_t)g.nqt * N, nQ = (size_t)g.npb * N;
    // bit 0: written, bit 1: carries a baseline, bit 2: read by creduce
    unsigned char* fp = new unsigned char[nP]();
    unsigned char* fq = new unsigned char[nQ]();
    int64_t live = 0;
    for (int qt = 0; qt < g.nqt; qt++) {
        for (int pb = 0; pb < g.npb; pb++) {
            const int q0 = CP_TQ * qt, qmax = (N < q0 + CP_TQ ? N : q0 + CP_TQ) - 1, p0 = CP_PB * pb;
            if (p0 >= qmax) continue;
            live++;
            for (int r = 0; r < CP_PB; r++) {
                const int p = p0 + r;
                if (p >= N - 1) break;
                fp[(size_t)qt * N + p] |= 1;
                for (int lane = 0; lane < CP_TQ; lane++) {
                    const int q = q0 + lane;
                    if (q > p && q < N) {
                        cover[bl_index(N, p, q)]++;
                        fp[(size_t)qt * N + p] |= 2;
                        fq[(size_t)pb * N + q] |= 2;
                    }
                }
            }
            for (int lane = 0; lane < CP_TQ; lane++)
                if (q0 + lane < N) fq[(size_t)pb * N + q0 + lane] |= 1;
        }
    }
    for (int s = 0; s < N; s++) {
        if (s <= N - 2)
            for (int qt = (s + 1) / CP_TQ; qt < g.nqt; qt++) fp[(size_t)qt * N + s] |= 4;
        if (s >= 1) {
            const int qmax = (N < CP_TQ * (s / CP_TQ) + CP_TQ ? N : CP_TQ * (s / CP_TQ) + CP_TQ) - 1;
            int npb = (qmax - 1) / CP_PB + 1;
            if (npb > g.npb) npb = g.npb;
            for (int pb = 0; pb < npb; pb++) fq[(size_t)pb * N + s] |= 4;
        }
    }
    int bad = 0;
    for (size_t i = 0; i < nP; i++) {
        if ((fp[i] & 4) && !(fp[i] & 1)) bad |= 1;   // read but never written
        if ((fp[i] & 2) && !(fp[i] & 4)) bad |= 2;   // carries a baseline but is not read
    }
    for (size_t i = 0; i < nQ; i++) {
        if ((fq[i] & 4) && !(fq[i] & 1)) bad |= 4;
        if ((fq[i] & 2) && !(fq[i] & 4)) bad |= 8;
    }
    delete[] fp;
    delete[] fq;
    info[0] = g.nqt; info[1] = g.npb; info[2] = live; info[3] = g.B;
    return bad;
}
