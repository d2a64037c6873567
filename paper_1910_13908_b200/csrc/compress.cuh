// Time/frequency-compressed M-step: shared declarations of wbstat.cu (per-baseline statistics,
// fused with the previous cluster's write-back) and mstep.cu (the LM iterations of one M-step on those statistics).
//
// One Jones matrix per (cluster, station) holds for the whole interval (reading Q7), so for a fixed
// baseline every (t, f) sample sees the same J_p, J_q.  With c = vec(C) (row-major [C00,C01,C10,C11]), r = vec(R)
// the residual at the centre Jones J0, and W(J) = J_p (x) conj(J_q)  (so vec(J_p C J_q^H) = W c):
//
//   E(J)  = r - dW c,                dW = W(J) - W(J0) = D_p (x) conj(J0_q) + J_p (x) conj(D_q),  D = J - J0
//   Src   = sum_tf r c^H  (4x4),     Scc = sum_tf c c^H (4x4 Hermitian),     srr = sum_tf |r|^2
//   Sec   = sum_tf E c^H = Src - dW Scc
//   cost  = srr - Re tr(dW^H (Src + Sec))
//   G_p[i,k] = sum_{j,l} J_q[j,l] Sec[(i,j),(k,l)]            G_q[j,l] = sum_{i,k} J_p[i,k] conj(Sec[(i,j),(k,l)])
//   M_p[k,k'] = sum_{l,l'} (J_q^H J_q)[l,l'] Scc[(k,l),(k',l')]   M_q[l,l'] = sum_{k,k'} (J_p^H J_p)[k,k'] conj(Scc[(k,l),(k',l')])
//
// which are sagecal_lm_cost_grad_jtj's sums (A5-A6) re-associated; nothing is approximated.  Statistics are taken of
// the RESIDUAL, not of the data, so the cancellation in `cost` is relative to the cost at the centre of the M-step.
// Scalar coherencies (C = c I2): Sr = sum conj(c) r (2x2), s2 = sum |c|^2, dP = D_p J0_q^H + J_p D_q^H,
//   Se = Sr - s2 dP, cost = srr - Re tr(dP^H (Sr + Se)), G_p = Se J_q, G_q = Se^H J_p, M_p = s2 J_q^H J_q, M_q = s2 J_p^H J_p.
#pragma once
#include "common.cuh"

namespace sgc {

// ---- statistics layout: one record per baseline ----------------------------------------------------------------
//   Src  FULL   [B][34]: [4 a][4 c] complex, Src[a][c] = sum r_a conj(c_c), then srr, then one pad (272 B)
//        SCALAR [B][10]: [4 a] complex Sr[a], then srr, then one pad (80 B)
//   Scc  [K][B][NSCC] doubles: FULL 16 = Scc[0][0], [1][1], [2][2], [3][3], then Re, Im of the upper pairs in the order
//        (0,1) (0,2) (0,3) (1,2) (1,3) (2,3)  (128 B);  SCALAR 1 = s2
constexpr int NSRC_FULL = 34, NSRC_SCALAR = 10;   // doubles per record; srr sits at index NSRC-2
constexpr int NSCC_FULL = 16, NSCC_SCALAR = 1;
__host__ __device__ constexpr int nsrc(bool scalar) { return scalar ? NSRC_SCALAR : NSRC_FULL; }
__host__ __device__ constexpr int nscc(bool scalar) { return scalar ? NSCC_SCALAR : NSCC_FULL; }

// lanes that share one baseline in wbstat/gram: the smallest power of two >= F, at most 32
inline int stat_group(int F) { int g = 1; while (g < F && g < 32) g <<= 1; return g; }

#ifdef __CUDACC__
// ---- entries of dW / dP from the centre and the current Jones (wbstat.cu, wbgroup.cu) -----------------------------
// dW[a][c] (a = 2i+j, c = 2k+l) = D_p[i,k] conj(J0_q[j,l]) + J_p[i,k] conj(D_q[j,l])
__device__ __forceinline__ cplx dW_entry(const sagecal_c128* __restrict__ J0, const sagecal_c128* __restrict__ J, int p,
                                         int q, int a, int c) {
    const int i = a >> 1, j = a & 1, k = c >> 1, l = c & 1;
    const sagecal_c128 jp0 = J0[4 * p + 2 * i + k], jp = J[4 * p + 2 * i + k];
    const sagecal_c128 jq0 = J0[4 * q + 2 * j + l], jq = J[4 * q + 2 * j + l];
    const cplx Dp = mk(jp.re - jp0.re, jp.im - jp0.im), Dq = mk(jq.re - jq0.re, jq.im - jq0.im);
    return cfmac(mk(jp.re, jp.im), Dq, cmulc(Dp, mk(jq0.re, jq0.im)));
}
// dP[a] (a = 2i+j) = (D_p J0_q^H + J_p D_q^H)[i,j]
__device__ __forceinline__ cplx dP_entry(const sagecal_c128* __restrict__ J0, const sagecal_c128* __restrict__ J, int p,
                                         int q, int a) {
    const int i = a >> 1, j = a & 1;
    cplx acc = mk(0.0, 0.0);
#pragma unroll
    for (int k = 0; k < 2; k++) {
        const sagecal_c128 jp0 = J0[4 * p + 2 * i + k], jp = J[4 * p + 2 * i + k];
        const sagecal_c128 jq0 = J0[4 * q + 2 * j + k], jq = J[4 * q + 2 * j + k];
        const cplx Dp = mk(jp.re - jp0.re, jp.im - jp0.im), Dq = mk(jq.re - jq0.re, jq.im - jq0.im);
        acc = cfmac(mk(jp.re, jp.im), Dq, cfmac(Dp, mk(jq0.re, jq0.im), acc));
    }
    return acc;
}

#endif

// ---- M-step kernel work decomposition (mstep.cu) -------------------------------------------------------------------
// One THREAD per baseline.  A unit is (column segment qt, row station p): the up to 32 baselines (p, q), q in
// [32 qt, 32 qt + 32), q > p, one per lane.  Segment qt has rows p = 0 .. nrows(qt)-1; units are numbered segment by
// segment, u = ubase(qt) + p.  A chunk is m consecutive rows of one segment and belongs to one warp for the whole
// launch (the lane's column station never changes, so its Jones and its column sums live in registers); chunks are
// numbered segment by segment too.  m is the smallest chunk length for which all chunks fit the co-resident warps.
constexpr int MS_THREADS = 256, MS_WARPS = 8, MS_TQ = 32, MS_NV = 12, MS_MAX_GRID = 160;
constexpr int MS_MAX_WARPS = MS_MAX_GRID * MS_WARPS;
struct MGeom {
    int N, nqt, m, nchunks, U;
    int64_t B;
    __host__ __device__ int nrows(int qt) const { int h = MS_TQ * (qt + 1); return (h < N ? h : N) - 1; }
    __host__ __device__ int chunks_in(int qt) const { return (nrows(qt) + m - 1) / m; }
    // units before segment qt (every earlier segment is full: 32 (t+1) - 1 rows)
    __host__ __device__ int ubase(int qt) const { return 16 * qt * (qt + 1) - qt; }
    // chunks before segment qt
    __host__ __device__ int cbase(int qt) const { int c = 0; for (int t = 0; t < qt; t++) c += chunks_in(t); return c; }
    // chunk c -> its segment, first row and number of rows
    __host__ __device__ void decode(int c, int& qt, int& p0, int& cnt) const {
        qt = 0;
        for (;;) { const int nc = chunks_in(qt); if (c < nc || qt == nqt - 1) break; c -= nc; qt++; }
        p0 = c * m;
        const int left = nrows(qt) - p0;
        cnt = left < m ? (left > 0 ? left : 0) : m;
    }
};
inline MGeom make_mgeom(int N, int max_warps) {
    MGeom g;
    g.N = N; g.nqt = (N + MS_TQ - 1) / MS_TQ; g.B = (int64_t)N * (N - 1) / 2;
    g.U = g.ubase(g.nqt - 1) + (N - 1);
    for (g.m = 1;; g.m++) {
        g.nchunks = g.cbase(g.nqt);
        if (g.nchunks <= max_warps) break;
    }
    return g;
}

// LM state carried between the chunks of one M-step (device memory)
struct MstepCtl { double phi, mu, nu, pad; };

struct CompressWorkspace {
    double* Scc;      // [K][B][nscc]
    double* Src;      // [B][nsrc]
    double* Ppart;    // [U][12]  row-station partial sums, one record per unit
    double* Qpart;    // [MS_MAX_WARPS][32][12]  column-station partial sums, one record per (chunk, column)
    double* cost_cta; // [MS_MAX_GRID] cost summed per CTA
    double* pred_cta; // [2][MS_MAX_GRID] predicted reduction summed per CTA, halves alternate by evaluation (readers
                      //        of one evaluation must not see the next one's values)
    double* mm_cta;   // [MS_MAX_GRID] max over the CTA's stations of max(M00, M11) (damping initialisation)
    sagecal_c128 *G, *M, *J_try;   // [N][4] accepted gradient / J^H J, trial Jones
    MstepCtl* ctl;
    unsigned* bar;    // grid barrier arrive counter (zeroed before every launch)
    sagecal_c128* J0; // [2][N][4] centre Jones of the current / previous statistics
    // cluster-group path (wbgroup.cu)
    double* SrcG;     // [GRP][B][nsrc] statistics of the GRP clusters of the current group
    double* Xg;       // [ngroups*GRP_PAIRS][B][nx] cross grams X_ij = sum_tf c_i c_j^H of the cluster pairs inside a group
    sagecal_c128* J0G;// [2][GRP][N][4] centre Jones of the clusters of the current / previous group
};
// ---- cluster groups (wbgroup.cu; DESIGN.md §5.5 "cluster groups") ---------------------------------------------------
// The statistics are linear in R, so the write-back of GRP consecutive clusters can be deferred and done in ONE pass
// over R together with the statistics of the next GRP clusters: Src_j taken of the stale residual is corrected per
// baseline by Src_j -= dW_i X_ij once cluster i < j of the same group has been solved.
constexpr int GRP = 4, GRP_PAIRS = GRP * (GRP - 1) / 2;
constexpr int NX_FULL = 32, NX_SCALAR = 2;
__host__ __device__ constexpr int nxg(bool scalar) { return scalar ? NX_SCALAR : NX_FULL; }
__host__ __device__ constexpr int grp_pair(int i, int j) { return i * GRP - i * (i + 1) / 2 + (j - i - 1); }   // i < j
inline int ngroups(int K) { return (K + GRP - 1) / GRP; }

// R -= sum_{i<gp} dW_i c_{kp0+i}, then Src of the new R against c_{kn0+j}, j < gn, into SrcG[j] (srr into SrcG[0] only).
// Scc != NULL (first EM iteration): also Scc of clusters kn0..kn0+gn-1 (into Scc + k*nscc*B) and the cross grams of
// their pairs (into Xgroup), by the GRAM arm of the same kernel.
int enqueue_wbgroup(int N, int T, int F, int coh_format, sagecal_c128* R, const sagecal_c128* coh, size_t cstride,
                    int kp0, int gp, const sagecal_c128* J0prev, const sagecal_c128* jones, int kn0, int gn,
                    double* SrcG, double* Scc, double* Xgroup, cudaStream_t st);
// right before cluster j >= 1 of the group is solved: Src_j -= sum_{i<j} dW_i X_ij and srr_j = cost per baseline after
// cluster j-1's update.  J0g / Jg: centre and solved Jones of the group's clusters ([GRP][N][4], [>= j][N][4]);
// Scc_prev: Scc of cluster j-1
int enqueue_groupfix(int N, bool scalar, int j, const sagecal_c128* J0g, const sagecal_c128* Jg, const double* Scc_prev,
                     const double* Xgroup, double* SrcG, cudaStream_t st);
size_t compress_workspace_bytes(int N, int K, bool scalar);
CompressWorkspace carve_compress(int N, int K, bool scalar, void* ws);

// R -= dW(J0prev -> Jprev) c_prev  (if Cprev), then the Src records (with srr) of the new R against Cnext (if Cnext),
// and Scc of Cnext into Scc_next if that is not NULL
int enqueue_wbstat(int N, int T, int F, int coh_format, sagecal_c128* R, const sagecal_c128* Cprev,
                   const sagecal_c128* J0prev, const sagecal_c128* Jprev, const sagecal_c128* Cnext, double* Src,
                   double* Scc_next, cudaStream_t st);
// One chunk of an M-step on the statistics, one cooperative launch: J0 <- Jk, evaluation at J0, then n_trial trial
// steps with the accept/reject and damping control on the device (init: damping initialised from tau, else the
// state in w.ctl continues).  Jk is updated in place; *cost_out (and *trace_out) receive the accepted cost.
int enqueue_mstep(int N, bool scalar, const CompressWorkspace& w, const double* Scc_k, sagecal_c128* J0,
                  sagecal_c128* Jk, int n_trial, bool init, double tau, double* cost_out, double* trace_out,
                  cudaStream_t st);

// lm_mode = SAGECAL_LM_FULLGN (fullgn.cu): one chunk of a full Gauss-Newton M-step on the same statistics; fgn_ws is
// device scratch of fullgn_workspace_bytes(N).
size_t fullgn_workspace_bytes(int N);
int enqueue_fullgn(int N, bool scalar, const CompressWorkspace& cw, const double* Scc_k, sagecal_c128* J0,
                   sagecal_c128* Jk, int n_trial, bool init, double tau, double* cost_out, double* trace_out,
                   void* fgn_ws, cudaStream_t st);

}  // namespace sgc
