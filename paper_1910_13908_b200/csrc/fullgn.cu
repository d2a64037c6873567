// lm_mode = SAGECAL_LM_FULLGN: the M-step with the FULL Gauss-Newton normal
// matrix -- the other reading of "per-station-block J^H J ... small dense per-cluster solve" (Q1): all 8N x 8N real
// entries, one off-diagonal 8x8 block per baseline, damped Cholesky solve with cuSOLVER.  Not the hot path: it exists
// for the reading's sake (an M-step converges in a handful of steps instead of ~45) and is written for clarity, one
// thread per baseline, on top of the same per-baseline statistics as the compressed mode (compress.cuh):
//
//   theta_p = [Re vec(J_p); Im vec(J_p)],   g = -Jac^T r = [Re vec(G_p); Im vec(G_p)]
//   H_pp = [[Re K, -Im K], [Im K, Re K]],  K = I2 (x) M_p^T                                        (A6)
//   H_pq = [[Re Z, Im Z], [Im Z, -Re Z]],  Z[(i,k),(j,l)] = sum_{m,n} J_q[j,m] J_p[i,n] conj(Scc[(k,m),(n,l)])
//          (from <d_p E, d_q E> = Re tr[(D_p C J_q^H)^H (J_p C D_q^H)] summed over t, f)
//   (H + mu I) delta = g,   J' = J + delta,   pred = delta^T (g + mu delta),   then the accept/reject rule of A7.
#include <cusolverDn.h>
#include <math.h>
#include "compress.cuh"

namespace sgc {

constexpr int FG_REC = 58;   // doubles per baseline record: cost, gp[8], gq[8], mp[4], mq[4], Z[32], pad
constexpr int FG_THREADS = 128;

struct FgnCtl { double phi, phi_try, mu, nu, pred; int accept; int pad; };

__device__ __forceinline__ cplx ldc(const sagecal_c128* p) { return mk(p->re, p->im); }
__device__ __forceinline__ cplx cconj_(cplx a) { return mk(a.re, -a.im); }

// ---- F1: one thread per baseline: cost, gradient and J^H J contributions and the off-diagonal block -------------
template <bool SCALAR>
__global__ void __launch_bounds__(FG_THREADS)
fgn_baseline_kernel(int N, int64_t B, const double* __restrict__ Src, const double* __restrict__ Scc,
                    const sagecal_c128* __restrict__ J0, const sagecal_c128* __restrict__ Jt, double* __restrict__ rec) {
    const int64_t b = (int64_t)blockIdx.x * FG_THREADS + threadIdx.x;
    if (b >= B) return;
    int p, q;
    bl_stations(N, b, p, q);
    cplx Jp[4], Jq[4], Dp[4], Dq[4], Jq0[4];
#pragma unroll
    for (int x = 0; x < 4; x++) {
        Jp[x] = ldc(Jt + 4 * p + x); Jq[x] = ldc(Jt + 4 * q + x); Jq0[x] = ldc(J0 + 4 * q + x);
        const cplx jp0 = ldc(J0 + 4 * p + x);
        Dp[x] = mk(Jp[x].re - jp0.re, Jp[x].im - jp0.im);
        Dq[x] = mk(Jq[x].re - Jq0[x].re, Jq[x].im - Jq0[x].im);
    }
    // H = J^H J as a full 2x2
    cplx Hp[4], Hq[4];
#pragma unroll
    for (int l = 0; l < 2; l++)
#pragma unroll
        for (int l2 = 0; l2 < 2; l2++) {
            Hp[2 * l + l2] = cfmaca(Jp[2 + l], Jp[2 + l2], cfmaca(Jp[l], Jp[l2], mk(0.0, 0.0)));
            Hq[2 * l + l2] = cfmaca(Jq[2 + l], Jq[2 + l2], cfmaca(Jq[l], Jq[l2], mk(0.0, 0.0)));
        }
    cplx gp[4], gq[4], mp[4], mq[4], Z[16];
#pragma unroll
    for (int x = 0; x < 4; x++) gp[x] = gq[x] = mp[x] = mq[x] = mk(0.0, 0.0);
    double cost;
    if (SCALAR) {
        const double* r = Src + b * NSRC_SCALAR;
        const double s2 = Scc[b];
        double acc = 0.0;
        cplx Se[4];
#pragma unroll
        for (int a = 0; a < 4; a++) {
            const int i = a >> 1, j = a & 1;
            cplx dP = mk(0.0, 0.0);
#pragma unroll
            for (int k = 0; k < 2; k++) dP = cfmac(Jp[2 * i + k], Dq[2 * j + k], cfmac(Dp[2 * i + k], Jq0[2 * j + k], dP));
            const cplx sr = mk(r[2 * a], r[2 * a + 1]);
            Se[a] = mk(fma(-s2, dP.re, sr.re), fma(-s2, dP.im, sr.im));
            acc = fma(dP.re, sr.re + Se[a].re, fma(dP.im, sr.im + Se[a].im, acc));
        }
        cost = r[NSRC_SCALAR - 2] - acc;
#pragma unroll
        for (int i = 0; i < 2; i++)
#pragma unroll
            for (int k = 0; k < 2; k++) {
                gp[2 * i + k] = cfma(Se[2 * i + 1], Jq[2 + k], cmul(Se[2 * i], Jq[k]));          // (Se J_q)[i,k]
                gq[2 * i + k] = cfmaca(Se[2 + i], Jp[2 + k], cfmaca(Se[i], Jp[k], mk(0.0, 0.0))); // (Se^H J_p)[i,k]
            }
#pragma unroll
        for (int x = 0; x < 4; x++) {
            mp[x] = mk(s2 * Hq[x].re, s2 * Hq[x].im);
            mq[x] = mk(s2 * Hp[x].re, s2 * Hp[x].im);
        }
        // Z[(i,k),(j,l)] = s2 J_q[j,k] J_p[i,l]
#pragma unroll
        for (int i = 0; i < 2; i++)
#pragma unroll
            for (int k = 0; k < 2; k++)
#pragma unroll
                for (int j = 0; j < 2; j++)
#pragma unroll
                    for (int l = 0; l < 2; l++) {
                        const cplx t = cmul(Jq[2 * j + k], Jp[2 * i + l]);
                        Z[4 * (2 * i + k) + 2 * j + l] = mk(s2 * t.re, s2 * t.im);
                    }
    } else {
        const double* sr = Src + b * NSRC_FULL;
        const double* sc = Scc + b * NSCC_FULL;
        cplx S[4][4];
        S[0][0] = mk(sc[0], 0.0); S[1][1] = mk(sc[1], 0.0); S[2][2] = mk(sc[2], 0.0); S[3][3] = mk(sc[3], 0.0);
        S[0][1] = mk(sc[4], sc[5]); S[0][2] = mk(sc[6], sc[7]); S[0][3] = mk(sc[8], sc[9]);
        S[1][2] = mk(sc[10], sc[11]); S[1][3] = mk(sc[12], sc[13]); S[2][3] = mk(sc[14], sc[15]);
#pragma unroll
        for (int x = 0; x < 4; x++)
#pragma unroll
            for (int y = x + 1; y < 4; y++) S[y][x] = cconj_(S[x][y]);
        double acc = 0.0;
#pragma unroll
        for (int a = 0; a < 4; a++) {
            const int i = a >> 1, j = a & 1;
            cplx dW[4], sec[4];
#pragma unroll
            for (int c = 0; c < 4; c++)
                dW[c] = cfmac(Jp[2 * i + (c >> 1)], Dq[2 * j + (c & 1)], cmulc(Dp[2 * i + (c >> 1)], Jq0[2 * j + (c & 1)]));
#pragma unroll
            for (int c = 0; c < 4; c++) {
                const cplx sv = mk(sr[2 * (4 * a + c)], sr[2 * (4 * a + c) + 1]);
                cplx t = sv;
#pragma unroll
                for (int d = 0; d < 4; d++) t = cfms(dW[d], S[d][c], t);
                sec[c] = t;
                acc = fma(dW[c].re, sv.re + t.re, fma(dW[c].im, sv.im + t.im, acc));
            }
#pragma unroll
            for (int k = 0; k < 2; k++) {
                gp[2 * i + k] = cfma(Jq[2 * j + 1], sec[2 * k + 1], cfma(Jq[2 * j], sec[2 * k], gp[2 * i + k]));
                gq[2 * j + k] = cfmac(Jp[2 * i + 1], sec[2 + k], cfmac(Jp[2 * i], sec[k], gq[2 * j + k]));
            }
        }
        cost = sr[NSRC_FULL - 2] - acc;
        // M_p[k,k'] = sum_{l,l'} Hq[l,l'] S[(k,l)][(k',l')];  M_q[l,l'] = sum_{k,k'} Hp[k,k'] conj(S[(k,l)][(k',l')])
#pragma unroll
        for (int k = 0; k < 2; k++)
#pragma unroll
            for (int k2 = 0; k2 < 2; k2++)
#pragma unroll
                for (int l = 0; l < 2; l++)
#pragma unroll
                    for (int l2 = 0; l2 < 2; l2++) {
                        mp[2 * k + k2] = cfma(Hq[2 * l + l2], S[2 * k + l][2 * k2 + l2], mp[2 * k + k2]);
                        mq[2 * l + l2] = cfmac(Hp[2 * k + k2], S[2 * k + l][2 * k2 + l2], mq[2 * l + l2]);
                    }
        // Z[(i,k),(j,l)] = sum_{m,n} J_q[j,m] J_p[i,n] conj(S[(k,m)][(n,l)])
#pragma unroll
        for (int i = 0; i < 2; i++)
#pragma unroll
            for (int k = 0; k < 2; k++)
#pragma unroll
                for (int j = 0; j < 2; j++)
#pragma unroll
                    for (int l = 0; l < 2; l++) {
                        cplx z = mk(0.0, 0.0);
#pragma unroll
                        for (int m = 0; m < 2; m++)
#pragma unroll
                            for (int n = 0; n < 2; n++)
                                z = cfmac(cmul(Jq[2 * j + m], Jp[2 * i + n]), S[2 * k + m][2 * n + l], z);
                        Z[4 * (2 * i + k) + 2 * j + l] = z;
                    }
    }
    double* o = rec + (size_t)b * FG_REC;
    o[0] = cost;
#pragma unroll
    for (int x = 0; x < 4; x++) {
        o[1 + 2 * x] = gp[x].re; o[2 + 2 * x] = gp[x].im;
        o[9 + 2 * x] = gq[x].re; o[10 + 2 * x] = gq[x].im;
    }
    o[17] = mp[0].re; o[18] = mp[3].re; o[19] = mp[1].re; o[20] = mp[1].im;
    o[21] = mq[0].re; o[22] = mq[3].re; o[23] = mq[1].re; o[24] = mq[1].im;
#pragma unroll
    for (int x = 0; x < 16; x++) { o[25 + 2 * x] = Z[x].re; o[26 + 2 * x] = Z[x].im; }
}

__device__ __forceinline__ double fg_block_sum(double v, double* s_buf) {   // fixed-order tree over FG_THREADS
    const int tid = threadIdx.x;
    s_buf[tid] = v;
    __syncthreads();
    for (int o = FG_THREADS / 2; o > 0; o >>= 1) {
        if (tid < o) s_buf[tid] += s_buf[tid + o];
        __syncthreads();
    }
    const double r = s_buf[0];
    __syncthreads();
    return r;
}
__device__ __forceinline__ double fg_block_max(double v, double* s_buf) {
    const int tid = threadIdx.x;
    s_buf[tid] = v;
    __syncthreads();
    for (int o = FG_THREADS / 2; o > 0; o >>= 1) {
        if (tid < o) s_buf[tid] = fmax(s_buf[tid], s_buf[tid + o]);
        __syncthreads();
    }
    const double r = s_buf[0];
    __syncthreads();
    return r;
}

// ---- F2: CTA s adds station s's records in a fixed order; writes G_try, M_try, cost_st and H's diagonal block -----
__global__ void __launch_bounds__(FG_THREADS)
fgn_assemble_kernel(int N, const double* __restrict__ rec, sagecal_c128* __restrict__ G, sagecal_c128* __restrict__ M,
                    double* __restrict__ cost_st, double* __restrict__ H) {
    __shared__ double s_buf[FG_THREADS];
    __shared__ double s_out[13];
    const int s = blockIdx.x, tid = threadIdx.x;
    double acc[13];
#pragma unroll
    for (int x = 0; x < 13; x++) acc[x] = 0.0;
    for (int o = tid; o < N; o += FG_THREADS) {
        if (o == s) continue;
        const bool row = s < o;                                   // s is the row station p of baseline (s, o)
        const double* r = rec + (size_t)(row ? bl_index(N, s, o) : bl_index(N, o, s)) * FG_REC;
        const double* gg = r + (row ? 1 : 9);
        const double* mm = r + (row ? 17 : 21);
#pragma unroll
        for (int x = 0; x < 8; x++) acc[x] += gg[x];
#pragma unroll
        for (int x = 0; x < 4; x++) acc[8 + x] += mm[x];
        if (row) acc[12] += r[0];
    }
    for (int x = 0; x < 13; x++) {
        const double v = fg_block_sum(acc[x], s_buf);
        if (tid == 0) s_out[x] = v;
    }
    __syncthreads();
    if (tid == 0) {
        for (int x = 0; x < 4; x++) { G[4 * s + x].re = s_out[2 * x]; G[4 * s + x].im = s_out[2 * x + 1]; }
        M[4 * s].re = s_out[8]; M[4 * s].im = 0.0;
        M[4 * s + 1].re = s_out[10]; M[4 * s + 1].im = s_out[11];
        M[4 * s + 2].re = s_out[10]; M[4 * s + 2].im = -s_out[11];
        M[4 * s + 3].re = s_out[9]; M[4 * s + 3].im = 0.0;
        cost_st[s] = s_out[12];
    }
    // diagonal block: K[(i,k),(i',k')] = delta_ii' M[k',k];  H_pp = [[Re K, -Im K], [Im K, Re K]]
    if (tid < 64) {
        const int r8 = tid >> 3, c8 = tid & 7;
        const int a = r8 & 3, bcol = c8 & 3;                      // a = (i,k), bcol = (i',k')
        double v = 0.0;
        if ((a >> 1) == (bcol >> 1)) {
            const int k = a & 1, k2 = bcol & 1;                   // M[k2][k]
            const double mre = k == k2 ? (k ? s_out[9] : s_out[8]) : s_out[10];
            const double mim = k == k2 ? 0.0 : (k2 < k ? s_out[11] : -s_out[11]);   // M[0][1] = (s10, s11), M[1][0] = conj
            const bool rim = r8 >= 4, cim = c8 >= 4;
            v = rim == cim ? mre : (rim ? mim : -mim);
        }
        const size_t n = (size_t)8 * N;
        H[(size_t)(8 * s + r8) * n + 8 * s + c8] = v;
    }
}

// ---- F3: off-diagonal blocks, one thread per (baseline, entry): H_pq = [[Re Z, Im Z], [Im Z, -Re Z]] and H_qp = H_pq^T
__global__ void __launch_bounds__(256)
fgn_offdiag_kernel(int N, int64_t B, const double* __restrict__ rec, double* __restrict__ H) {
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= B * 64) return;
    const int64_t b = i >> 6;
    const int e = (int)(i & 63), r8 = e >> 3, c8 = e & 7;
    int p, q;
    bl_stations(N, b, p, q);
    const double* z = rec + (size_t)b * FG_REC + 25 + 2 * (4 * (r8 & 3) + (c8 & 3));
    const bool rim = r8 >= 4, cim = c8 >= 4;
    const double v = rim == cim ? (rim ? -z[0] : z[0]) : z[1];
    const size_t n = (size_t)8 * N;
    H[(size_t)(8 * p + r8) * n + 8 * q + c8] = v;
    H[(size_t)(8 * q + c8) * n + 8 * p + r8] = v;
}

// ---- F4: Hw = H + mu I, rhs = g = [Re vec G; Im vec G] -------------------------------------------------------------
__global__ void __launch_bounds__(256)
fgn_prep_kernel(int N, const double* __restrict__ H, const sagecal_c128* __restrict__ G, const FgnCtl* __restrict__ ctl,
                double* __restrict__ Hw, double* __restrict__ rhs) {
    const size_t n = (size_t)8 * N, total = n * n;
    const double mu = ctl->mu;
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < total; i += (size_t)gridDim.x * 256) {
        const size_t r = i / n, c = i - r * n;
        Hw[i] = H[i] + (r == c ? mu : 0.0);
        if (i < n) {
            const int s = (int)(i >> 3), x = (int)(i & 7);
            rhs[i] = x < 4 ? G[4 * s + x].re : G[4 * s + x - 4].im;
        }
    }
}

// ---- F5: J_try = J + delta, pred = delta^T (g + mu delta) ------------------------------------------------------------
__global__ void __launch_bounds__(FG_THREADS)
fgn_step_kernel(int N, const double* __restrict__ delta, const sagecal_c128* __restrict__ J,
                const sagecal_c128* __restrict__ G, sagecal_c128* __restrict__ J_try, FgnCtl* __restrict__ ctl) {
    __shared__ double s_buf[FG_THREADS];
    const double mu = ctl->mu;
    double part = 0.0;
    for (int s = threadIdx.x; s < N; s += FG_THREADS) {
#pragma unroll
        for (int x = 0; x < 4; x++) {
            const double dr = delta[8 * s + x], di = delta[8 * s + 4 + x];
            J_try[4 * s + x].re = J[4 * s + x].re + dr;
            J_try[4 * s + x].im = J[4 * s + x].im + di;
            part += dr * (G[4 * s + x].re + mu * dr) + di * (G[4 * s + x].im + mu * di);
        }
    }
    const double pred = fg_block_sum(part, s_buf);
    if (threadIdx.x == 0) ctl->pred = pred;
}

// ---- F6: LM control.  MODE 1 init (mu from tau), 2 re-centre (mu, nu kept), 0 trial (rho test) ------------------------
template <int MODE>
__global__ void __launch_bounds__(FG_THREADS)
fgn_control_kernel(int N, double tau, FgnCtl* __restrict__ ctl, const double* __restrict__ cost_st,
                   sagecal_c128* __restrict__ J, const sagecal_c128* __restrict__ J_try, sagecal_c128* __restrict__ G,
                   const sagecal_c128* __restrict__ G_try, sagecal_c128* __restrict__ M,
                   const sagecal_c128* __restrict__ M_try, const int* __restrict__ info, double* __restrict__ cost_out,
                   double* __restrict__ trace_out) {
    __shared__ double s_buf[FG_THREADS];
    const int tid = threadIdx.x;
    double part = 0.0;
    for (int s = tid; s < N; s += FG_THREADS) part += cost_st[s];
    const double fresh = fg_block_sum(part, s_buf);
    double phi = ctl->phi, mu = ctl->mu, nu = ctl->nu;
    bool accept = true;
    if (MODE == 1) {
        double mmax = 0.0;
        for (int s = tid; s < N; s += FG_THREADS) mmax = fmax(mmax, fmax(M_try[4 * s].re, M_try[4 * s + 3].re));
        mu = tau * fg_block_max(mmax, s_buf);
        nu = 2.0;
        phi = fresh;
    } else if (MODE == 2) {
        phi = fresh;
    } else {
        const double pred = ctl->pred, rho = (phi - fresh) / pred;
        // a Cholesky factorisation that broke down (H + mu I numerically indefinite: H has four gauge null directions)
        // leaves a partial factor and a meaningless step: reject it, the damping grows
        accept = isfinite(fresh) && isfinite(pred) && isfinite(rho) && pred > 0.0 && rho > 0.0 && info[0] == 0 && info[1] == 0;
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
    if (accept) {
        for (int i = tid; i < 4 * N; i += FG_THREADS) {
            G[i] = G_try[i];
            M[i] = M_try[i];
            if (MODE == 0) J[i] = J_try[i];
        }
    }
    if (tid == 0) {
        ctl->phi = phi; ctl->mu = mu; ctl->nu = nu; ctl->accept = accept ? 1 : 0;
        if (cost_out) *cost_out = phi;
        if (trace_out) *trace_out = phi;
    }
}

// ---- F7: H_acc <- H_try if the last control step accepted ------------------------------------------------------------
__global__ void __launch_bounds__(256)
fgn_commit_kernel(size_t total, const FgnCtl* __restrict__ ctl, const double* __restrict__ H_try, double* __restrict__ H) {
    if (!ctl->accept) return;
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < total; i += (size_t)gridDim.x * 256) H[i] = H_try[i];
}

// ---- host side ----------------------------------------------------------------------------------------------------
struct FgnWorkspace {
    double *H, *H_try, *Hw;        // [8N][8N]
    double *rec;                   // [B][FG_REC]
    double *rhs, *cost_st;         // [8N], [N]
    sagecal_c128 *G, *M, *G_try, *M_try, *J_try;
    FgnCtl* ctl;
    int* info;
};
size_t fullgn_workspace_bytes(int N) {
    const size_t n = (size_t)8 * N, B = (size_t)N * (N - 1) / 2;
    return 3 * round_up(sizeof(double) * n * n, 256) + round_up(sizeof(double) * B * FG_REC, 256) +
           round_up(sizeof(double) * n, 256) + round_up(sizeof(double) * (size_t)N, 256) +
           5 * round_up((size_t)N * 64, 256) + 256 + 256;
}
static FgnWorkspace carve_fullgn(int N, void* ws) {
    const size_t n = (size_t)8 * N, B = (size_t)N * (N - 1) / 2;
    FgnWorkspace w;
    char* p = (char*)ws;
    auto take = [&](size_t bytes) { char* o = p; p += round_up(bytes, 256); return o; };
    w.H = (double*)take(sizeof(double) * n * n);
    w.H_try = (double*)take(sizeof(double) * n * n);
    w.Hw = (double*)take(sizeof(double) * n * n);
    w.rec = (double*)take(sizeof(double) * B * FG_REC);
    w.rhs = (double*)take(sizeof(double) * n);
    w.cost_st = (double*)take(sizeof(double) * (size_t)N);
    w.G = (sagecal_c128*)take((size_t)N * 64);
    w.M = (sagecal_c128*)take((size_t)N * 64);
    w.G_try = (sagecal_c128*)take((size_t)N * 64);
    w.M_try = (sagecal_c128*)take((size_t)N * 64);
    w.J_try = (sagecal_c128*)take((size_t)N * 64);
    w.ctl = (FgnCtl*)take(256);
    w.info = (int*)take(256);
    return w;
}

static int cusolver_handle(cusolverDnHandle_t* out) {
    // a cuSOLVER handle is bound to the device that was current when it was created: one per (host thread, device)
    static thread_local cusolverDnHandle_t h[64] = {};
    int dev = 0;
    SGC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return SAGECAL_EUNSUPPORTED;
    if (!h[dev] && cusolverDnCreate(&h[dev]) != CUSOLVER_STATUS_SUCCESS) { h[dev] = nullptr; return cuda_fail(cudaErrorUnknown); }
    *out = h[dev];
    return SAGECAL_OK;
}

// evaluation at w.J_try from the statistics centred at J0: records, station sums, H_try
static int fgn_evaluate(int N, bool scalar, const CompressWorkspace& cw, const double* Scc_k, const sagecal_c128* J0,
                        const FgnWorkspace& w, cudaStream_t st) {
    const int64_t B = (int64_t)N * (N - 1) / 2;
    {
        LaunchScope ls(KK_FULLGN, st);
        const unsigned grid = (unsigned)((B + FG_THREADS - 1) / FG_THREADS);
        if (scalar) fgn_baseline_kernel<true><<<grid, FG_THREADS, 0, st>>>(N, B, cw.Src, Scc_k, J0, w.J_try, w.rec);
        else fgn_baseline_kernel<false><<<grid, FG_THREADS, 0, st>>>(N, B, cw.Src, Scc_k, J0, w.J_try, w.rec);
        SGC_LAUNCH_CHECK();
    }
    {
        LaunchScope ls(KK_FULLGN, st);
        fgn_assemble_kernel<<<N, FG_THREADS, 0, st>>>(N, w.rec, w.G_try, w.M_try, w.cost_st, w.H_try);
        SGC_LAUNCH_CHECK();
    }
    {
        LaunchScope ls(KK_FULLGN, st);
        fgn_offdiag_kernel<<<(unsigned)((B * 64 + 255) / 256), 256, 0, st>>>(N, B, w.rec, w.H_try);
        SGC_LAUNCH_CHECK();
    }
    return SAGECAL_OK;
}

// One chunk of a full Gauss-Newton M-step on the statistics in cw (centre J0 <- Jk, evaluation, n_trial trial steps).
int enqueue_fullgn(int N, bool scalar, const CompressWorkspace& cw, const double* Scc_k, sagecal_c128* J0,
                   sagecal_c128* Jk, int n_trial, bool init, double tau, double* cost_out, double* trace_out,
                   void* fgn_ws, cudaStream_t st) {
    const FgnWorkspace w = carve_fullgn(N, fgn_ws);
    const int n = 8 * N;
    const size_t total = (size_t)n * n;
    const unsigned gs = (unsigned)(total / 256 < 2048 ? (total + 255) / 256 : 2048);
    cusolverDnHandle_t h;
    int rc;
    if ((rc = cusolver_handle(&h))) return rc;
    if (cusolverDnSetStream(h, st) != CUSOLVER_STATUS_SUCCESS) return cuda_fail(cudaErrorUnknown);
    int lwork = 0;
    if (cusolverDnDpotrf_bufferSize(h, CUBLAS_FILL_MODE_LOWER, n, w.Hw, n, &lwork) != CUSOLVER_STATUS_SUCCESS)
        return cuda_fail(cudaErrorUnknown);
    double* work = nullptr;                 // cuSOLVER's scratch: its size is only known with a device, so it is
    SGC_CUDA(cudaMallocAsync((void**)&work, sizeof(double) * (size_t)(lwork > 0 ? lwork : 1), st));   // stream-ordered
    // from here on every exit path frees `work`
    auto chk = [&](cudaError_t e) { if (!rc && e != cudaSuccess) rc = cuda_fail(e); };
    chk(cudaMemcpyAsync(J0, Jk, (size_t)N * 64, cudaMemcpyDeviceToDevice, st));
    chk(cudaMemcpyAsync(w.J_try, Jk, (size_t)N * 64, cudaMemcpyDeviceToDevice, st));
    if (init) chk(cudaMemsetAsync(w.ctl, 0, sizeof(FgnCtl), st));
    chk(cudaMemsetAsync(w.info, 0, 2 * sizeof(int), st));
    if (!rc) rc = fgn_evaluate(N, scalar, cw, Scc_k, J0, w, st);
    if (!rc) {
        LaunchScope ls(KK_FULLGN, st);
        if (init)
            fgn_control_kernel<1><<<1, FG_THREADS, 0, st>>>(N, tau, w.ctl, w.cost_st, Jk, w.J_try, w.G, w.G_try, w.M, w.M_try, w.info, cost_out, trace_out);
        else
            fgn_control_kernel<2><<<1, FG_THREADS, 0, st>>>(N, tau, w.ctl, w.cost_st, Jk, w.J_try, w.G, w.G_try, w.M, w.M_try, w.info, cost_out, trace_out);
        if (cudaGetLastError() != cudaSuccess) rc = cuda_fail(cudaErrorLaunchFailure);
    }
    if (!rc) {
        LaunchScope ls(KK_FULLGN, st);
        fgn_commit_kernel<<<gs, 256, 0, st>>>(total, w.ctl, w.H_try, w.H);
    }
    for (int i = 0; i < n_trial && !rc; i++) {
        {
            LaunchScope ls(KK_FULLGN, st);
            fgn_prep_kernel<<<gs, 256, 0, st>>>(N, w.H, w.G, w.ctl, w.Hw, w.rhs);
        }
        if (cusolverDnDpotrf(h, CUBLAS_FILL_MODE_LOWER, n, w.Hw, n, work, lwork, w.info) != CUSOLVER_STATUS_SUCCESS ||
            cusolverDnDpotrs(h, CUBLAS_FILL_MODE_LOWER, n, 1, w.Hw, n, w.rhs, n, w.info + 1) != CUSOLVER_STATUS_SUCCESS) {
            rc = cuda_fail(cudaErrorUnknown);
            break;
        }
        {
            LaunchScope ls(KK_FULLGN, st);
            fgn_step_kernel<<<1, FG_THREADS, 0, st>>>(N, w.rhs, Jk, w.G, w.J_try, w.ctl);
        }
        if ((rc = fgn_evaluate(N, scalar, cw, Scc_k, J0, w, st))) break;
        {
            LaunchScope ls(KK_FULLGN, st);
            fgn_control_kernel<0><<<1, FG_THREADS, 0, st>>>(N, tau, w.ctl, w.cost_st, Jk, w.J_try, w.G, w.G_try, w.M, w.M_try, w.info, cost_out, trace_out);
        }
        {
            LaunchScope ls(KK_FULLGN, st);
            fgn_commit_kernel<<<gs, 256, 0, st>>>(total, w.ctl, w.H_try, w.H);
        }
        if (cudaGetLastError() != cudaSuccess) rc = cuda_fail(cudaErrorLaunchFailure);
    }
    const cudaError_t ef = cudaFreeAsync(work, st);
    if (!rc && ef != cudaSuccess) rc = cuda_fail(ef);
    return rc;
}

}  // namespace sgc
