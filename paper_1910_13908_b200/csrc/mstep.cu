// One chunk of a compressed M-step as ONE cooperative kernel (formulas: compress.cuh): the initial
// evaluation at the centre Jones and n_trial Levenberg-Marquardt trial steps, each = cost / gradient / per-station
// J^H J from the per-baseline statistics (rows 8a-4, 8a-5 of SURVEY.md §8(a) re-associated), with the damping,
// accept/reject and 2x2 solves on the device and grid-wide barriers between the phases:
//
//   A  tiles   : CTA <- tile (PB row stations p x 32 column stations q); 4 lanes share one baseline, lane a = 2i+j
//                owns row a of dW / Sec, i.e. residual entry (i, j): it needs only row i of J_p and row j of J_q.
//                Row-station sums: shuffles over the lanes, combined over the 4 warps of a row in shared memory,
//                one record per (column tile, row).  Column-station sums: registers over the rows, combined over
//                the 2 row groups in shared memory, one record per (row block, column).  Cost: one sum per CTA.
//      -- grid barrier --
//   B  control : every warp adds the CTA costs and the stations' predicted reductions in the same fixed order
//                (identical in all CTAs), takes the accept/reject decision and updates mu, nu.  Warp <-> station:
//                adds the station's records (lanes over records, butterfly), commits or discards the trial, solves
//                dJ_p = G_p (M_p + mu I)^-1, writes the next trial Jones, its Gram matrix and predicted reduction.
//      -- grid barrier --
//
// No atomics, fixed summation order: bit-reproducible for a given grid.  The statistics (392 B per baseline, 51 MB
// at N=512) stay L2-resident over the evaluations.
#include <cooperative_groups.h>
#include <math.h>
#include "compress.cuh"

namespace cg = cooperative_groups;

namespace sgc {

struct MstepArgs {
    MGeom g;
    const double *Src, *srr, *Scc;
    double *Ppart, *Qpart, *cost_cta, *pred_st, *mm_st, *Htry;
    sagecal_c128 *G, *M, *J_try, *J0, *Jk;
    MstepCtl* ctl;
    int n_trial, init;
    double tau;
    double *cost_out, *trace_out;
};

__device__ __forceinline__ double wsum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ cplx ldcg_c(const sagecal_c128* p) {   // coherent at L2: data other CTAs write
    const double2 v = __ldcg(reinterpret_cast<const double2*>(p));
    return mk(v.x, v.y);
}
__device__ __forceinline__ void st_c(sagecal_c128* p, cplx v) { p->re = v.re; p->im = v.im; }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return mk(a.re - b.re, a.im - b.im); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return mk(a.re + b.re, a.im + b.im); }

// every lane of every warp gets the same sum: lane-strided partial sums, then a butterfly
__device__ __forceinline__ double strided_sum(const double* p, int n, int lane) {
    double v = 0.0;
    for (int i = lane; i < n; i += 32) v += __ldcg(p + i);
    return wsum(v);
}
__device__ __forceinline__ double strided_max(const double* p, int n, int lane) {
    double v = 0.0;
    for (int i = lane; i < n; i += 32) v = fmax(v, __ldcg(p + i));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

struct Herm { double h00, h11; cplx h01; };
__device__ __forceinline__ Herm load_herm(const double* H, int s) {
    const double2 a = __ldcg(reinterpret_cast<const double2*>(H + 4 * s));
    const double2 b = __ldcg(reinterpret_cast<const double2*>(H + 4 * s + 2));
    Herm h; h.h00 = a.x; h.h11 = a.y; h.h01 = mk(b.x, b.y);
    return h;
}

// ---- one lane's share of one baseline -----------------------------------------------------------------------------
// lane a = 2i+j.  jp, dp: row i of the trial J_p and of D_p;  jq, jq0, dq: row j of the trial J_q, of J0_q, of D_q.
// gp += its part of G_p row i;  gqc = its part of G_q row j;  mp / mq: a=0 (M_p00, M_p11), a=1 M_p01, a=2 (M_q00, M_q11),
// a=3 M_q01.
template <bool SCALAR>
__device__ __forceinline__ void lane_task(const double* __restrict__ Src, const double* __restrict__ srr,
                                          const double* __restrict__ Scc, int64_t b, int a, const cplx* jp,
                                          const cplx* dp, const cplx* jq, const cplx* jq0, const cplx* dq,
                                          const Herm& hp, const Herm& hq, cplx* gp, cplx* gqc, double* mp, double* mq,
                                          double& cost) {
    if (SCALAR) {
        const double s2 = __ldg(Scc + b);
        const cplx sr = ldg128_stream(Src + b * NSRC_SCALAR + 2 * a);
        // dP[(i,j)] = sum_k D_p[i,k] conj(J0_q[j,k]) + J_p[i,k] conj(D_q[j,k])
        cplx dP = cmulc(dp[0], jq0[0]);
        dP = cfmac(dp[1], jq0[1], dP);
        dP = cfmac(jp[0], dq[0], dP);
        dP = cfmac(jp[1], dq[1], dP);
        const cplx se = mk(fma(-s2, dP.re, sr.re), fma(-s2, dP.im, sr.im));
        const double acc = fma(dP.re, sr.re + se.re, dP.im * (sr.im + se.im));
        cost += (a == 0 ? __ldg(srr + b) : 0.0) - acc;
        gp[0] = cfma(se, jq[0], gp[0]);           // G_p[i,k] += Se[(i,j)] J_q[j,k]
        gp[1] = cfma(se, jq[1], gp[1]);
        gqc[0] = cmulc(jp[0], se);                // G_q[j,l] += conj(Se[(i,j)]) J_p[i,l]
        gqc[1] = cmulc(jp[1], se);
        if (a == 0) { mp[0] = fma(s2, hq.h00, mp[0]); mp[1] = fma(s2, hq.h11, mp[1]); }
        else if (a == 1) { mp[0] = fma(s2, hq.h01.re, mp[0]); mp[1] = fma(s2, hq.h01.im, mp[1]); }
        else if (a == 2) { mq[0] = fma(s2, hp.h00, mq[0]); mq[1] = fma(s2, hp.h11, mq[1]); }
        else { mq[0] = fma(s2, hp.h01.re, mq[0]); mq[1] = fma(s2, hp.h01.im, mq[1]); }
        return;
    }
    // Hermitian Scc: 128 B record
    const double* sp = Scc + b * NSCC_FULL;
    const d4 s0 = ldg256_stream(sp), s1 = ldg256_stream(sp + 4), s2 = ldg256_stream(sp + 8), s3 = ldg256_stream(sp + 12);
    cplx S[4][4];
    S[0][0] = mk(s0.x, 0.0); S[1][1] = mk(s0.y, 0.0); S[2][2] = mk(s0.z, 0.0); S[3][3] = mk(s0.w, 0.0);
    S[0][1] = mk(s1.x, s1.y); S[0][2] = mk(s1.z, s1.w); S[0][3] = mk(s2.x, s2.y);
    S[1][2] = mk(s2.z, s2.w); S[1][3] = mk(s3.x, s3.y); S[2][3] = mk(s3.z, s3.w);
#pragma unroll
    for (int x = 0; x < 4; x++) {
#pragma unroll
        for (int y = x + 1; y < 4; y++) S[y][x] = mk(S[x][y].re, -S[x][y].im);
    }
    // row a of Src: 64 B
    const double* rp = Src + b * NSRC_FULL + 8 * a;
    const d4 r0 = ldg256_stream(rp), r1 = ldg256_stream(rp + 4);
    const cplx src[4] = {mk(r0.x, r0.y), mk(r0.z, r0.w), mk(r1.x, r1.y), mk(r1.z, r1.w)};
    // row a of dW: dW[(k,l)] = D_p[i,k] conj(J0_q[j,l]) + J_p[i,k] conj(D_q[j,l])
    cplx dW[4];
#pragma unroll
    for (int c = 0; c < 4; c++) dW[c] = cfmac(jp[c >> 1], dq[c & 1], cmulc(dp[c >> 1], jq0[c & 1]));
    cplx sec[4];
    double acc = 0.0;
#pragma unroll
    for (int c = 0; c < 4; c++) {
        cplx s = src[c];
#pragma unroll
        for (int d = 0; d < 4; d++) s = cfms(dW[d], S[d][c], s);
        sec[c] = s;
        acc = fma(dW[c].re, src[c].re + s.re, fma(dW[c].im, src[c].im + s.im, acc));
    }
    cost += (a == 0 ? __ldg(srr + b) : 0.0) - acc;
    // G_p[i,k] += sum_l J_q[j,l] Sec[(i,j),(k,l)];   G_q[j,l] += sum_k J_p[i,k] conj(Sec[(i,j),(k,l)])
    gp[0] = cfma(jq[1], sec[1], cfma(jq[0], sec[0], gp[0]));
    gp[1] = cfma(jq[1], sec[3], cfma(jq[0], sec[2], gp[1]));
    gqc[0] = cfmac(jp[1], sec[2], cmulc(jp[0], sec[0]));
    gqc[1] = cfmac(jp[1], sec[3], cmulc(jp[0], sec[1]));
    if (a == 0) {          // M_p[k,k] = sum_{l,l'} Hq[l,l'] S[(k,l)][(k,l')]
        mp[0] += fma(hq.h00, S[0][0].re, fma(hq.h11, S[1][1].re, 2.0 * fma(hq.h01.re, S[0][1].re, -hq.h01.im * S[0][1].im)));
        mp[1] += fma(hq.h00, S[2][2].re, fma(hq.h11, S[3][3].re, 2.0 * fma(hq.h01.re, S[2][3].re, -hq.h01.im * S[2][3].im)));
    } else if (a == 1) {   // M_p[0,1] = Hq00 S[0][2] + Hq01 S[0][3] + conj(Hq01) S[1][2] + Hq11 S[1][3]
        cplx m = mk(hq.h00 * S[0][2].re, hq.h00 * S[0][2].im);
        m = cfma(hq.h01, S[0][3], m);
        m = cfmaca(hq.h01, S[1][2], m);
        mp[0] += fma(hq.h11, S[1][3].re, m.re);
        mp[1] += fma(hq.h11, S[1][3].im, m.im);
    } else if (a == 2) {   // M_q[l,l] = sum_{k,k'} Hp[k,k'] conj(S[(k,l)][(k',l)])
        mq[0] += fma(hp.h00, S[0][0].re, fma(hp.h11, S[2][2].re, 2.0 * fma(hp.h01.re, S[0][2].re, hp.h01.im * S[0][2].im)));
        mq[1] += fma(hp.h00, S[1][1].re, fma(hp.h11, S[3][3].re, 2.0 * fma(hp.h01.re, S[1][3].re, hp.h01.im * S[1][3].im)));
    } else {               // M_q[0,1] = Hp00 conj(S[0][1]) + Hp01 conj(S[0][3]) + conj(Hp01) S[1][2] + Hp11 conj(S[2][3])
        cplx m = mk(hp.h00 * S[0][1].re, -hp.h00 * S[0][1].im);
        m = cfmac(hp.h01, S[0][3], m);
        m = cfmaca(hp.h01, S[1][2], m);
        mq[0] += fma(hp.h11, S[2][3].re, m.re);
        mq[1] += fma(-hp.h11, S[2][3].im, m.im);
    }
}

// ---- phase A ------------------------------------------------------------------------------------------------------
template <bool SCALAR>
__device__ __forceinline__ void phase_tiles(const MstepArgs& A, double (*s_p)[4][MS_NV], double (*s_q)[MS_TQ][MS_NV],
                                            double* s_cost) {
    const MGeom& g = A.g;
    const int N = g.N, PB = g.PB;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int sq = warp & 3, rg = warp >> 2;
    const int qi = lane >> 2, a = lane & 3, i = a >> 1, j = a & 1;
    double cost = 0.0;
    for (int tile = blockIdx.x; tile < g.ntiles; tile += gridDim.x) {
        int qt = 0, pb = tile;
        while (pb >= g.nlive(qt)) { pb -= g.nlive(qt); qt++; }
        const int q = MS_TQ * qt + 8 * sq + qi, qc = min(q, N - 1);
        cplx jq[2], jq0[2], dq[2];
#pragma unroll
        for (int l = 0; l < 2; l++) {
            jq[l] = ldcg_c(A.J_try + 4 * qc + 2 * j + l);
            jq0[l] = ldcg_c(A.J0 + 4 * qc + 2 * j + l);
            dq[l] = csub(jq[l], jq0[l]);
        }
        const Herm hq = load_herm(A.Htry, qc);
        cplx gq[2] = {mk(0.0, 0.0), mk(0.0, 0.0)};
        double mq[2] = {0.0, 0.0};
        for (int r = rg; r < PB; r += 2) {
            const int p = PB * pb + r;
            if (p >= N - 1) break;                                  // warp-uniform
            cplx jp[2], dp[2];
#pragma unroll
            for (int k = 0; k < 2; k++) {
                jp[k] = ldcg_c(A.J_try + 4 * p + 2 * i + k);
                dp[k] = csub(jp[k], ldcg_c(A.J0 + 4 * p + 2 * i + k));
            }
            const Herm hp = load_herm(A.Htry, p);
            cplx gp[2] = {mk(0.0, 0.0), mk(0.0, 0.0)}, gqc[2] = {mk(0.0, 0.0), mk(0.0, 0.0)};
            double mp[2] = {0.0, 0.0};
            if (q < N && q > p)
                lane_task<SCALAR>(A.Src, A.srr, A.Scc, bl_index(N, p, q), a, jp, dp, jq, jq0, dq, hp, hq, gp, gqc, mp, mq, cost);
            // row station: G_p row i over j (xor 1) and the 8 columns (xor 4, 8, 16); M slots over the columns
            double v[6] = {gp[0].re, gp[0].im, gp[1].re, gp[1].im, mp[0], mp[1]};
#pragma unroll
            for (int x = 0; x < 4; x++) v[x] += __shfl_xor_sync(0xffffffffu, v[x], 1);
#pragma unroll
            for (int o = 4; o <= 16; o <<= 1) {
#pragma unroll
                for (int x = 0; x < 6; x++) v[x] += __shfl_xor_sync(0xffffffffu, v[x], o);
            }
            if (qi == 0) {
                double* rec = s_p[r][sq];
                if (a == 0) { rec[0] = v[0]; rec[1] = v[1]; rec[2] = v[2]; rec[3] = v[3]; rec[8] = v[4]; rec[9] = v[5]; }
                else if (a == 1) { rec[10] = v[4]; rec[11] = v[5]; }
                else if (a == 2) { rec[4] = v[0]; rec[5] = v[1]; rec[6] = v[2]; rec[7] = v[3]; }
            }
            // column station: G_q row j over i (xor 2), accumulated over the rows
#pragma unroll
            for (int l = 0; l < 2; l++) {
                gq[l].re += gqc[l].re + __shfl_xor_sync(0xffffffffu, gqc[l].re, 2);
                gq[l].im += gqc[l].im + __shfl_xor_sync(0xffffffffu, gqc[l].im, 2);
            }
        }
        {
            double* rec = s_q[rg][8 * sq + qi];
            if (a == 0) { rec[0] = gq[0].re; rec[1] = gq[0].im; rec[2] = gq[1].re; rec[3] = gq[1].im; }
            else if (a == 1) { rec[4] = gq[0].re; rec[5] = gq[0].im; rec[6] = gq[1].re; rec[7] = gq[1].im; }
            else if (a == 2) { rec[8] = mq[0]; rec[9] = mq[1]; }
            else { rec[10] = mq[0]; rec[11] = mq[1]; }
        }
        __syncthreads();
        for (int o = tid; o < PB * MS_NV; o += MS_THREADS) {
            const int r = o / MS_NV, x = o - r * MS_NV, p = PB * pb + r;
            if (p < N - 1)
                A.Ppart[((size_t)qt * N + p) * MS_NV + x] = ((s_p[r][0][x] + s_p[r][1][x]) + s_p[r][2][x]) + s_p[r][3][x];
        }
        for (int o = tid; o < MS_TQ * MS_NV; o += MS_THREADS) {
            const int ql = o / MS_NV, x = o - ql * MS_NV, qq = MS_TQ * qt + ql;
            if (qq < N) A.Qpart[((size_t)pb * N + qq) * MS_NV + x] = s_q[0][ql][x] + s_q[1][ql][x];
        }
        __syncthreads();
    }
    cost = wsum(cost);
    if (lane == 0) s_cost[warp] = cost;
    __syncthreads();
    if (tid == 0) {
        double c = s_cost[0];
#pragma unroll
        for (int w = 1; w < MS_WARPS; w++) c += s_cost[w];
        A.cost_cta[blockIdx.x] = c;
    }
}

// ---- phase B helpers ----------------------------------------------------------------------------------------------
struct StAcc { cplx g[4]; cplx m[4]; };

// adds station s's records: lanes over records, butterfly; every lane returns the sums
__device__ __forceinline__ StAcc station_reduce(const MstepArgs& A, int s, int lane) {
    const MGeom& g = A.g;
    const int N = g.N;
    double acc[MS_NV];
#pragma unroll
    for (int x = 0; x < MS_NV; x++) acc[x] = 0.0;
    if (s <= N - 2) {
        for (int qt = (s + 1) / MS_TQ + lane; qt < g.nqt; qt += 32) {
            const double* rec = A.Ppart + ((size_t)qt * N + s) * MS_NV;
#pragma unroll
            for (int x = 0; x < MS_NV; x++) acc[x] += __ldcg(rec + x);
        }
    }
    if (s >= 1) {
        const int nl = g.nlive(s / MS_TQ);
        for (int pb = lane; pb < nl; pb += 32) {
            const double* rec = A.Qpart + ((size_t)pb * N + s) * MS_NV;
#pragma unroll
            for (int x = 0; x < MS_NV; x++) acc[x] += __ldcg(rec + x);
        }
    }
#pragma unroll
    for (int x = 0; x < MS_NV; x++) acc[x] = wsum(acc[x]);
    StAcc r;
#pragma unroll
    for (int x = 0; x < 4; x++) r.g[x] = mk(acc[2 * x], acc[2 * x + 1]);
    r.m[0] = mk(acc[8], 0.0); r.m[1] = mk(acc[10], acc[11]); r.m[2] = mk(acc[10], -acc[11]); r.m[3] = mk(acc[9], 0.0);
    return r;
}

// dJ = G (M + mu I)^-1, J_try = J + dJ; returns this station's predicted reduction Re tr(G^H dJ) + mu ||dJ||^2
__device__ __forceinline__ double trial_step(const MstepArgs& A, int s, int lane, const cplx* g, const cplx* m,
                                             const cplx* jj, double mu, double* pred_out) {
    const double a = m[0].re + mu, d = m[3].re + mu;
    const cplx b = m[1];
    const double det = a * d - (b.re * b.re + b.im * b.im);
    const cplx inv[4] = {mk(d / det, 0.0), mk(-b.re / det, -b.im / det), mk(-b.re / det, b.im / det), mk(a / det, 0.0)};
    cplx dj[4], jt[4];
    dj[0] = cfma(g[1], inv[2], cmul(g[0], inv[0]));
    dj[1] = cfma(g[1], inv[3], cmul(g[0], inv[1]));
    dj[2] = cfma(g[3], inv[2], cmul(g[2], inv[0]));
    dj[3] = cfma(g[3], inv[3], cmul(g[2], inv[1]));
    double pred = 0.0;
#pragma unroll
    for (int x = 0; x < 4; x++) {
        jt[x] = cadd(jj[x], dj[x]);
        pred += g[x].re * dj[x].re + g[x].im * dj[x].im;
        pred += mu * (dj[x].re * dj[x].re + dj[x].im * dj[x].im);
    }
    if (lane == 0) {
#pragma unroll
        for (int x = 0; x < 4; x++) st_c(A.J_try + 4 * s + x, jt[x]);
        // H = J_try^H J_try
        A.Htry[4 * s] = cabs2(jt[2], cabs2(jt[0], 0.0));
        A.Htry[4 * s + 1] = cabs2(jt[3], cabs2(jt[1], 0.0));
        const cplx h01 = cfmaca(jt[2], jt[3], cfmaca(jt[0], jt[1], mk(0.0, 0.0)));
        A.Htry[4 * s + 2] = h01.re;
        A.Htry[4 * s + 3] = h01.im;
        pred_out[s] = pred;
    }
    return pred;
}

template <bool SCALAR>
__global__ void __launch_bounds__(MS_THREADS, 2)
mstep_kernel(const MstepArgs A) {
    __shared__ double s_p[MS_PB_MAX][4][MS_NV];
    __shared__ double s_q[2][MS_TQ][MS_NV];
    __shared__ double s_cost[MS_WARPS];
    cg::grid_group grid = cg::this_grid();
    const int N = A.g.N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gw = blockIdx.x * MS_WARPS + warp, nw = gridDim.x * MS_WARPS;

    // LM state, identical in every thread of the grid
    double phi = 0.0, mu = A.init ? 0.0 : A.ctl->mu, nu = A.init ? 2.0 : A.ctl->nu;

    // prologue: centre and first "trial" = the current Jones of the cluster
    for (int s = gw; s < N; s += nw) {
        cplx jj[4];
#pragma unroll
        for (int x = 0; x < 4; x++) jj[x] = ldcg_c(A.Jk + 4 * s + x);
        if (lane == 0) {
#pragma unroll
            for (int x = 0; x < 4; x++) { st_c(A.J0 + 4 * s + x, jj[x]); st_c(A.J_try + 4 * s + x, jj[x]); }
            A.Htry[4 * s] = cabs2(jj[2], cabs2(jj[0], 0.0));
            A.Htry[4 * s + 1] = cabs2(jj[3], cabs2(jj[1], 0.0));
            const cplx h01 = cfmaca(jj[2], jj[3], cfmaca(jj[0], jj[1], mk(0.0, 0.0)));
            A.Htry[4 * s + 2] = h01.re;
            A.Htry[4 * s + 3] = h01.im;
        }
    }
    grid.sync();

    for (int e = 0; e <= A.n_trial; e++) {
        phase_tiles<SCALAR>(A, s_p, s_q, s_cost);
        grid.sync();

        const double fresh = strided_sum(A.cost_cta, (int)gridDim.x, lane);
        bool accept = false;
        if (e == 0) {
            phi = fresh;
            if (A.init) {
                // (phi, G, M) at the centre are the accepted state; mu = tau * max_p max(M_p00, M_p11)
                for (int s = gw; s < N; s += nw) {
                    const StAcc r = station_reduce(A, s, lane);
                    if (lane == 0) {
#pragma unroll
                        for (int x = 0; x < 4; x++) { st_c(A.G + 4 * s + x, r.g[x]); st_c(A.M + 4 * s + x, r.m[x]); }
                        A.mm_st[s] = fmax(r.m[0].re, r.m[3].re);
                    }
                }
                grid.sync();
                mu = A.tau * strided_max(A.mm_st, N, lane);
                nu = 2.0;
            }
        } else {
            // written by the stations' owners in the previous evaluation; this evaluation's go to the other half
            const double pred = strided_sum(A.pred_st + (size_t)((e - 1) & 1) * N, N, lane);
            const double rho = (phi - fresh) / pred;
            accept = isfinite(fresh) && isfinite(pred) && isfinite(rho) && pred > 0.0 && rho > 0.0;
            if (accept) {
                phi = fresh;
                const double t = 2.0 * rho - 1.0;
                mu *= fmax(1.0 / 3.0, 1.0 - t * t * t);
                nu = 2.0;
            } else {
                mu *= nu;
                nu *= 2.0;
            }
        }
        if (!(mu >= 1e-300)) mu = 1e-300;
        if (mu > 1e300) mu = 1e300;
        if (nu > 0x1p60) nu = 0x1p60;

        const bool last = e == A.n_trial;
        for (int s = gw; s < N; s += nw) {
            cplx g4[4], m4[4], jj[4];
            if (e == 0 && A.init) {
#pragma unroll
                for (int x = 0; x < 4; x++) { g4[x] = ldcg_c(A.G + 4 * s + x); m4[x] = ldcg_c(A.M + 4 * s + x); jj[x] = ldcg_c(A.Jk + 4 * s + x); }
            } else {
                // speculative loads of the accepted state, in flight while the records are added
                cplx go[4], mo[4], jo[4], jt[4];
#pragma unroll
                for (int x = 0; x < 4; x++) {
                    go[x] = ldcg_c(A.G + 4 * s + x); mo[x] = ldcg_c(A.M + 4 * s + x);
                    jo[x] = ldcg_c(A.Jk + 4 * s + x); jt[x] = ldcg_c(A.J_try + 4 * s + x);
                }
                const StAcc r = station_reduce(A, s, lane);
                const bool take = accept || e == 0;       // e == 0 (re-centre): fresh (G, M) at the accepted Jones
#pragma unroll
                for (int x = 0; x < 4; x++) {
                    g4[x] = take ? r.g[x] : go[x];
                    m4[x] = take ? r.m[x] : mo[x];
                    jj[x] = accept ? jt[x] : jo[x];
                }
                if (take && lane == 0) {
#pragma unroll
                    for (int x = 0; x < 4; x++) {
                        st_c(A.G + 4 * s + x, g4[x]); st_c(A.M + 4 * s + x, m4[x]);
                        if (accept) st_c(A.Jk + 4 * s + x, jj[x]);
                    }
                }
            }
            if (!last) trial_step(A, s, lane, g4, m4, jj, mu, A.pred_st + (size_t)(e & 1) * N);
        }
        if (!last) grid.sync();
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        A.ctl->phi = phi; A.ctl->mu = mu; A.ctl->nu = nu;
        if (A.cost_out) *A.cost_out = phi;
        if (A.trace_out) *A.trace_out = phi;
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------
// Rows per tile: the largest of 16, 8, 4, 2 that still gives about one tile per CTA slot of a B200 (148 SMs x 2);
// device independent, so the workspace can be sized without a device.
static int choose_pb(int N) {
    for (int PB = MS_PB_MAX; PB > 2; PB >>= 1)
        if (make_mgeom(N, PB).ntiles >= 252) return PB;
    return 2;
}

size_t compress_workspace_bytes(int N, int K, bool scalar) {
    const MGeom g = make_mgeom(N, choose_pb(N));
    size_t n = 0;
    n += round_up(sizeof(double) * (size_t)(K > 0 ? K : 1) * nscc(scalar) * g.B, 256);
    n += round_up(sizeof(double) * (size_t)nsrc(scalar) * g.B, 256);
    n += round_up(sizeof(double) * (size_t)g.B, 256);
    n += round_up(sizeof(double) * (size_t)g.nqt * N * MS_NV, 256);
    n += round_up(sizeof(double) * (size_t)g.npb * N * MS_NV, 256);
    n += round_up(sizeof(double) * MS_MAX_GRID, 256);
    n += round_up(sizeof(double) * 2 * (size_t)N, 256) + round_up(sizeof(double) * (size_t)N, 256);
    n += round_up(sizeof(double) * 4 * (size_t)N, 256);
    n += 3 * round_up((size_t)N * 64, 256);
    n += 256;
    n += round_up((size_t)2 * N * 64, 256);
    return n;
}

CompressWorkspace carve_compress(int N, int K, bool scalar, void* ws) {
    const MGeom g = make_mgeom(N, choose_pb(N));
    CompressWorkspace w;
    char* p = (char*)ws;
    auto take = [&](size_t n) { char* o = p; p += round_up(n, 256); return o; };
    w.Scc = (double*)take(sizeof(double) * (size_t)(K > 0 ? K : 1) * nscc(scalar) * g.B);
    w.Src = (double*)take(sizeof(double) * (size_t)nsrc(scalar) * g.B);
    w.srr = (double*)take(sizeof(double) * (size_t)g.B);
    w.Ppart = (double*)take(sizeof(double) * (size_t)g.nqt * N * MS_NV);
    w.Qpart = (double*)take(sizeof(double) * (size_t)g.npb * N * MS_NV);
    w.cost_cta = (double*)take(sizeof(double) * MS_MAX_GRID);
    w.pred_st = (double*)take(sizeof(double) * 2 * (size_t)N);
    w.mm_st = (double*)take(sizeof(double) * (size_t)N);
    w.Htry = (double*)take(sizeof(double) * 4 * (size_t)N);
    w.G = (sagecal_c128*)take((size_t)N * 64);
    w.M = (sagecal_c128*)take((size_t)N * 64);
    w.J_try = (sagecal_c128*)take((size_t)N * 64);
    w.ctl = (MstepCtl*)take(256);
    w.J0 = (sagecal_c128*)take((size_t)2 * N * 64);
    return w;
}

template <bool SCALAR>
static int max_coresident(int* out) {
    static int cached = 0;
    if (!cached) {
        int occ = 0;
        SGC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, mstep_kernel<SCALAR>, MS_THREADS, 0));
        if (occ < 1) return cuda_fail(cudaErrorLaunchOutOfResources);
        cached = occ * num_sms();
    }
    *out = cached;
    return SAGECAL_OK;
}

int enqueue_mstep(int N, bool scalar, const CompressWorkspace& w, const double* Scc_k, sagecal_c128* J0,
                  sagecal_c128* Jk, int n_trial, bool init, double tau, double* cost_out, double* trace_out,
                  cudaStream_t st) {
    MstepArgs A;
    A.g = make_mgeom(N, choose_pb(N));
    A.Src = w.Src; A.srr = w.srr; A.Scc = Scc_k;
    A.Ppart = w.Ppart; A.Qpart = w.Qpart; A.cost_cta = w.cost_cta; A.pred_st = w.pred_st; A.mm_st = w.mm_st; A.Htry = w.Htry;
    A.G = w.G; A.M = w.M; A.J_try = w.J_try; A.J0 = J0; A.Jk = Jk;
    A.ctl = w.ctl; A.n_trial = n_trial; A.init = init ? 1 : 0; A.tau = tau;
    A.cost_out = cost_out; A.trace_out = trace_out;
    int cap = 0, rc;
    if ((rc = scalar ? max_coresident<true>(&cap) : max_coresident<false>(&cap))) return rc;
    int grid = A.g.ntiles < cap ? A.g.ntiles : cap;
    if (grid > MS_MAX_GRID) grid = MS_MAX_GRID;
    if (grid < 1) grid = 1;
    void* args[] = {(void*)&A};
    LaunchScope ls(KK_MSTEP, st);
    SGC_CUDA(cudaLaunchCooperativeKernel(scalar ? (const void*)mstep_kernel<true> : (const void*)mstep_kernel<false>,
                                         dim3((unsigned)grid), dim3(MS_THREADS), args, 0, st));
    return SAGECAL_OK;
}

}  // namespace sgc

using namespace sgc;

// Host-side replay of the M-step kernel's tiling, lane mapping and record lists (CPU tests, no device needed).
extern "C" int sagecal_debug_mstep_cover(int N, int32_t* cover, int64_t* info) {
    if (N < 2 || !cover || !info) return SAGECAL_EINVAL;
    const MGeom g = make_mgeom(N, choose_pb(N));
    const int PB = g.PB;
    const size_t nP = (size_t)g.nqt * N, nQ = (size_t)g.npb * N;
    // bit 0: written, bit 1: carries a baseline, bit 2: read by the station reduction
    unsigned char* fp = new unsigned char[nP]();
    unsigned char* fq = new unsigned char[nQ]();
    int bad = 0;
    int64_t seen = 0;
    for (int tile = 0; tile < g.ntiles; tile++) {
        int qt = 0, pb = tile;
        while (qt < g.nqt && pb >= g.nlive(qt)) { pb -= g.nlive(qt); qt++; }
        if (qt >= g.nqt || pb >= g.npb) { bad |= 16; continue; }
        seen++;
        for (int warp = 0; warp < MS_WARPS; warp++) {
            const int sq = warp & 3, rg = warp >> 2;
            for (int r = rg; r < PB; r += 2) {
                const int p = PB * pb + r;
                if (p >= N - 1) break;
                fp[(size_t)qt * N + p] |= 1;
                for (int qi = 0; qi < 8; qi++) {
                    const int q = MS_TQ * qt + 8 * sq + qi;
                    if (q < N && q > p) {
                        cover[bl_index(N, p, q)]++;
                        fp[(size_t)qt * N + p] |= 2;
                        fq[(size_t)pb * N + q] |= 2;
                    }
                }
            }
        }
        for (int ql = 0; ql < MS_TQ; ql++)
            if (MS_TQ * qt + ql < N) fq[(size_t)pb * N + MS_TQ * qt + ql] |= 1;
    }
    for (int s = 0; s < N; s++) {
        if (s <= N - 2)
            for (int qt = (s + 1) / MS_TQ; qt < g.nqt; qt++) fp[(size_t)qt * N + s] |= 4;
        if (s >= 1)
            for (int pb = 0; pb < g.nlive(s / MS_TQ); pb++) {
                if (pb >= g.npb) { bad |= 32; break; }
                fq[(size_t)pb * N + s] |= 4;
            }
    }
    for (size_t x = 0; x < nP; x++) {
        if ((fp[x] & 4) && !(fp[x] & 1)) bad |= 1;   // read but never written
        if ((fp[x] & 2) && !(fp[x] & 4)) bad |= 2;   // carries a baseline but is not read
    }
    for (size_t x = 0; x < nQ; x++) {
        if ((fq[x] & 4) && !(fq[x] & 1)) bad |= 4;
        if ((fq[x] & 2) && !(fq[x] & 4)) bad |= 8;
    }
    delete[] fp;
    delete[] fq;
    info[0] = g.nqt; info[1] = g.npb; info[2] = seen; info[3] = g.B; info[4] = PB; info[5] = g.ntiles;
    return bad;
}
