// Time/frequency-compressed M-step: shared declarations of wbstat.cu (per-baseline statistics,
// fused with the previous cluster's write-back) and cpass.cu (cost / gradient / J^H J from those statistics).
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

// ---- statistics layout: structure of arrays over baselines, plane-major ---------------------------------------
//   Src [NSRC][B] doubles: FULL plane 2*(4a+b) = Re, +1 = Im of Src[a][b];  SCALAR plane 2a, 2a+1 of Sr[a]
//   srr [B]
//   Scc [K][NSCC][B]:      FULL planes 0..3 = Scc[a][a]; planes 4+2i, 5+2i = Re, Im of the i-th upper pair in the order
//                          (0,1) (0,2) (0,3) (1,2) (1,3) (2,3);  SCALAR plane 0 = s2
constexpr int NSRC_FULL = 32, NSRC_SCALAR = 8;
constexpr int NSCC_FULL = 16, NSCC_SCALAR = 1;
__host__ __device__ constexpr int nsrc(bool scalar) { return scalar ? NSRC_SCALAR : NSRC_FULL; }
__host__ __device__ constexpr int nscc(bool scalar) { return scalar ? NSCC_SCALAR : NSCC_FULL; }

// lanes that share one baseline in wbstat/gram: the smallest power of two >= F, at most 32
inline int stat_group(int F) { int g = 1; while (g < F && g < 32) g <<= 1; return g; }

// ---- compressed pass tiling: q tiles of 32 stations (one lane each) x p blocks of 16 rows ------------------------
constexpr int CP_TQ = 32, CP_PB = 16, CP_THREADS = 128, CP_NP = 13, CP_NQ = 12;
struct CGeom {
    int N, nqt, npb;
    int64_t B;
};
inline CGeom make_cgeom(int N) {
    CGeom g;
    g.N = N; g.nqt = (N + CP_TQ - 1) / CP_TQ; g.npb = (N - 1 + CP_PB - 1) / CP_PB;
    g.B = (int64_t)N * (N - 1) / 2;
    return g;
}

struct CompressWorkspace {
    double* Scc;      // [K][nscc][B]
    double* Src;      // [nsrc][B]
    double* srr;      // [B]
    double* Ppart;    // [nqt][N][13]  row-station partial sums (12 + cost)
    double* Qpart;    // [npb][N][12]  column-station partial sums
    double* cost_st;  // [N] cost summed per row station
    sagecal_c128* J0; // [2][N][4] centre Jones of the current / previous statistics
};
size_t compress_workspace_bytes(int N, int K, bool scalar);
CompressWorkspace carve_compress(int N, int K, bool scalar, void* ws);

// Scc of all K clusters (one pass over the coherencies)
int enqueue_gram(int N, int T, int F, int K, int coh_format, const sagecal_c128* coh, double* Scc, cudaStream_t st);
// R -= dW(J0prev -> Jprev) c_prev  (if Cprev), then Src, srr of the new R against Cnext (if Cnext)
int enqueue_wbstat(int N, int T, int F, int coh_format, sagecal_c128* R, const sagecal_c128* Cprev,
                   const sagecal_c128* J0prev, const sagecal_c128* Jprev, const sagecal_c128* Cnext, double* Src,
                   double* srr, cudaStream_t st);
// (cost_st, grad, jtj) at the trial Jones Jt from the statistics centred at J0
int enqueue_cpass(const CGeom& g, const CompressWorkspace& w, bool scalar, const double* Scc_k, const sagecal_c128* J0,
                  const sagecal_c128* Jt, sagecal_c128* grad, sagecal_c128* jtj, cudaStream_t st);

}  // namespace sgc
