// sagecal_predict_coherencies: point-source coherency prediction.
//
//   C_k[r][c] = sum_s B_s(f_c) exp(-2 pi i (f_c/c0)(u_r l_s + v_r m_s + w_r (n_s-1)))         (BASELINE.json:5)
//
// FP64-pipe bound.  One thread owns one uvw row and a register tile of FT channels; the cluster's sources are
// staged through shared memory in tiles and broadcast to the whole CTA.  For uniformly spaced channels the phasor
// of channel c+1 is the phasor of channel c times exp(-2 pi i ph df/c0): two sincospi per (row, source, channel
// tile) instead of FT, re-anchored at every tile so the recurrence never runs longer than FT-1 steps (one complex
// product, then the three-term form e_{c+1} = 2 cos(theta) e_c - e_{c-1}: error growth <= (FT-1)^2 eps = 5e-15).
// The phase is kept in cycles, so range reduction is exact: x = k/64 + r with k = rint(64 x) (magic-number rounding)
// and |r| <= 1/128 computed by one fma; exp(-2 pi i k/64) comes from a 64-entry table in shared memory and
// sin/cos(2 pi r) from degree-7/8 Taylor polynomials in r (remainders 5e-18 / 2e-20): 16 FP64 instructions per phasor
// against ~29 for sincospi(), same accuracy (a few 1e-16 absolute).
// precision = 1 (MIXED): the phase in cycles and its range reduction x - rint(x) stay in
// float64 (phases reach 3.3e3 cycles: float32 would leave 1e-4 cycles), then the phasor (sin.approx / cos.approx),
// the channel recurrence and the flux products run in float32; products are summed in float32 over at most 32 sources
// and those partial sums are added to the float64 accumulators.  Error ~2e-6 relative; the parity bound is 1e-5
// (BASELINE.json:5).
#include <mutex>
#include "common.cuh"

namespace sgc {

constexpr int PRED_THREADS = 128;
constexpr int PRED_MAXF = 512;
constexpr int PRED_MAXK = 1024;
constexpr int PRED_RPT = 2;           // rows per thread of the unpolarised float64 prediction (predict2_kernel)

struct PredFreqs { double kf[PRED_MAXF]; };          // f_c / c0  [1/m]
struct PredClusters { int off[PRED_MAXK + 1]; };

// ---- 8a-0: source-table preparation ---------------------------------------------------------------------------
// nm1[s] = -(l^2+m^2)/(1+sqrt(1-l^2-m^2));  flux[s][c][NFL] = (f_c/f0)^alpha_s * {I} or {I+Q, I-Q, U, V}
template <int NFL>
__global__ void predict_prep_kernel(int S, int F, int Fpad, PredFreqs fr, double c0_over_f0,
                                    const double* __restrict__ l, const double* __restrict__ m,
                                    const double* __restrict__ sI, const double* __restrict__ sQ,
                                    const double* __restrict__ sU, const double* __restrict__ sV,
                                    const double* __restrict__ alpha, double* __restrict__ nm1,
                                    double* __restrict__ flux) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S * Fpad) return;
    int s = i / Fpad, c = i - s * Fpad;
    if (c == 0) {
        double r2 = fma(l[s], l[s], m[s] * m[s]);
        nm1[s] = -r2 / (1.0 + sqrt(1.0 - r2));
    }
    double sc = (c < F) ? pow(fr.kf[c] * c0_over_f0, alpha[s]) : 0.0;  // padded channels contribute nothing
    double* o = flux + (size_t)i * NFL;
    if (NFL == 1) {
        o[0] = sc * sI[s];
    } else {
        o[0] = sc * (sI[s] + sQ[s]);
        o[1] = sc * (sI[s] - sQ[s]);
        o[2] = sc * sU[s];
        o[3] = sc * sV[s];
    }
}

// ---- 8a-1: the predict kernel ---------------------------------------------------------------------------------
// FT      channels per register tile
// POL     polarised sources (4 flux values, general 2x2 output) / unpolarised (C = c*I2)
// UNIFORM channel recurrence / one sincospi per channel
// SCALAR  output format SAGECAL_COH_SCALAR (only with !POL)
// MIXED   float32 phasors and products (precision = 1)
// exp(-2 pi i x), x in cycles; tab[8 k + c] = (cos, sin)(2 pi k/64) for c = 0..7: eight copies side by side, and
// `tab` already points at this lane's copy (lane & 7), so the 8 lanes of a quarter-warp read 8 different 16-byte
// columns of shared memory whatever their k: no bank conflicts (a single copy cost 1.8e9 conflict wavefronts per
// cfg4 launch and left the FP64 pipe at 61 %).
// The polynomial coefficients live in constant memory: a DFMA takes a constant-bank operand for free, whereas literal
// doubles were re-materialised by ~20 move instructions per loop trip, each of which costs the scheduler an issue slot
// the FP64 pipe's two-slot instructions leave it few of.
// PHC[0..3] = s1, s3, s5, s7 (sin(2 pi r) = r (s1 + s3 r^2 + ...)), PHC[4..7] = c2, c4, c6, c8, PHC[8] = 1.5 * 2^52
__constant__ double PHC[9] = {6.283185307179586476925286766559, -41.341702240399760233968420089468,
                              81.605249276075054203397682678249, -76.705859753061385841630641093893,
                              -19.739208802178717237668981999752, 64.939394022668291490960221297352,
                              -85.456817206693725260701221782482, 60.244641371876660575590717312223,
                              6755399441055744.0};
// `tab` is the BYTE address (shared window) of this lane's copy of entry 0: entry k sits 128 k bytes further.
__device__ __forceinline__ void phasor_f64(double x, unsigned tab, double& er, double& ei) {
    const double MAGIC = PHC[8];                                 // adding it rounds to the nearest integer
    double kd = fma(x, 64.0, MAGIC);
    const unsigned k = (unsigned)__double2loint(kd);
    kd -= MAGIC;
    const double r = fma(kd, -0.015625, x);                      // exact: |r| <= 1/128 cycle
    const double r2 = r * r;
    const double sp = r * fma(r2, fma(r2, fma(r2, PHC[3], PHC[2]), PHC[1]), PHC[0]);             // sin(2 pi r)
    const double cp = fma(r2, fma(r2, fma(r2, fma(r2, PHC[7], PHC[6]), PHC[5]), PHC[4]), 1.0);   // cos(2 pi r)
    double tx, ty;
    asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(tx), "=d"(ty) : "r"(tab + ((k << 7) & 0x1f80u)));
    er = fma(-ty, sp, tx * cp);                                  // cos(a + b)
    ei = -fma(tx, sp, ty * cp);                                  // -sin(a + b)
}
// float32 phasor of the MIXED arm: exact reduction to |r| <= 1/2 cycle in float64 (magic-number rounding: three DADDs,
// no FRND.F64), then the hardware approximations sin.approx / cos.approx (MUFU) on 2 pi r in [-pi, pi], where their
// absolute error is 2^-21.4 / 2^-21.2: configs[4] 20.9 ms with 1.7e-6 relative error against 25.7 ms / 5.8e-7 with
// sincospif (only the first channel's phasor from MUFU: 23.6 ms / 6.8e-7); the parity bound is 1e-5.
__device__ __forceinline__ void phasor_f32(double cycles, float& er, float& ei) {   // exp(-2 pi i cycles)
    const double MAGIC = PHC[8];
    const double kd = (cycles + MAGIC) - MAGIC;              // rint(cycles) for |cycles| < 2^51
    const float a = 6.283185307179586f * (float)(cycles - kd);
    er = __cosf(a); ei = -__sinf(a);
}
// RESID (sagecal_predict_residual): the CTA loops ALL clusters for its 128 rows, and next to writing C_k it takes
// R = V - sum_k J_k,p C_k J_k,q^H along: the rows' residual tile (FT channels x 4 correlations per thread) sits in
// shared memory, so R is written once and the initial residual pass over the K coherencies (69.7 GB at configs[4])
// is not needed.  Costs the prediction 16 (polarised: 64) more FP64 instructions per (row, cluster, channel).
struct PredResid { int N, K; int64_t B; const sagecal_c128 *jones, *vis; sagecal_c128* residual; };
template <int FT, bool POL, bool UNIFORM, bool SCALAR, bool MIXED, bool RESID>
__global__ void __launch_bounds__(PRED_THREADS)
predict_kernel(int64_t rows, int F, int Fpad, PredFreqs fr, double dkf, PredClusters cl,
               const double* __restrict__ uvw, const double* __restrict__ src_l,
               const double* __restrict__ src_m, const double* __restrict__ nm1_g,
               const double* __restrict__ flux_g, sagecal_c128* __restrict__ coh, PredResid rs) {
    extern __shared__ __align__(16) unsigned char s_dyn[];       // RESID: double2 [FT * 4][PRED_THREADS]
    double2* s_res = reinterpret_cast<double2*>(s_dyn) + threadIdx.x;
    constexpr int NFL = POL ? 4 : 1;
    constexpr int NACC = POL ? 4 : 1;            // complex accumulators per channel
    constexpr int ST = POL ? 32 : 128;           // sources per shared-memory tile
    __shared__ double s_l[ST], s_m[ST], s_n[ST];
    __shared__ __align__(16) double s_fl[MIXED ? 1 : ST * FT * NFL];
    __shared__ __align__(16) float s_flf[MIXED ? ST * FT * NFL : 1];
    __shared__ double2 s_tab_all[MIXED ? 1 : 64 * 8];
    if (!MIXED && threadIdx.x < 64) {
        double sn, cs;
        sincospi((double)threadIdx.x * 0.03125, &sn, &cs);       // 2 pi k/64 = pi k/32
#pragma unroll
        for (int c = 0; c < 8; c++) s_tab_all[8 * threadIdx.x + c] = make_double2(cs, sn);
    }
    const unsigned s_tab = (unsigned)__cvta_generic_to_shared(s_tab_all + (MIXED ? 0 : (threadIdx.x & 7)));

    const int64_t r = (int64_t)blockIdx.x * PRED_THREADS + threadIdx.x;
    const bool live = r < rows;
    double u = 0, v = 0, w = 0;
    if (live) { u = uvw[3 * r]; v = uvw[3 * r + 1]; w = uvw[3 * r + 2]; }
    int sp = 0, sq = 1;                                         // RESID: the row's stations
    if (RESID && live) bl_stations(rs.N, r % rs.B, sp, sq);
    const int k_begin = RESID ? 0 : blockIdx.y, k_end = RESID ? rs.K : k_begin + 1;

    for (int c0 = 0; c0 < Fpad; c0 += FT) {
      if (RESID && live) {
#pragma unroll
          for (int c = 0; c < FT; c++) {
              if (c0 + c < F) {
                  const sagecal_c128* vi = rs.vis + ((size_t)r * F + c0 + c) * 4;
                  const d4 lo = ldg256_stream(vi), hi = ldg256_stream(vi + 2);
                  s_res[(4 * c) * PRED_THREADS] = make_double2(lo.x, lo.y); s_res[(4 * c + 1) * PRED_THREADS] = make_double2(lo.z, lo.w);
                  s_res[(4 * c + 2) * PRED_THREADS] = make_double2(hi.x, hi.y); s_res[(4 * c + 3) * PRED_THREADS] = make_double2(hi.z, hi.w);
              }
          }
      }
      for (int k = k_begin; k < k_end; k++) {
        const int s_begin = cl.off[k], s_end = cl.off[k + 1];
        cplx acc[FT][NACC];
#pragma unroll
        for (int c = 0; c < FT; c++)
#pragma unroll
            for (int j = 0; j < NACC; j++) acc[c][j] = mk(0.0, 0.0);

        for (int sb = s_begin; sb < s_end; sb += ST) {
            const int ns = min(ST, s_end - sb);
            __syncthreads();
            for (int i = threadIdx.x; i < ns; i += PRED_THREADS) {
                s_l[i] = src_l[sb + i]; s_m[i] = src_m[sb + i]; s_n[i] = nm1_g[sb + i];
            }
            for (int i = threadIdx.x; i < ns * FT * NFL; i += PRED_THREADS) {
                int s = i / (FT * NFL), rem = i - s * (FT * NFL);
                const double f = flux_g[((size_t)(sb + s) * Fpad + c0) * NFL + rem];
                if (MIXED) s_flf[i] = (float)f; else s_fl[i] = f;
            }
            __syncthreads();
            if (MIXED) {
                for (int s0 = 0; s0 < ns; s0 += 32) {
                    float fr_[FT][NACC], fi_[FT][NACC];
#pragma unroll
                    for (int c = 0; c < FT; c++)
#pragma unroll
                        for (int j = 0; j < NACC; j++) fr_[c][j] = fi_[c][j] = 0.0f;
                    const int s1 = min(ns, s0 + 32);
#pragma unroll 2
                    for (int s = s0; s < s1; s++) {
                        const double ph = fma(w, s_n[s], fma(v, s_m[s], u * s_l[s]));  // metres
                        const float* fl = s_flf + s * (FT * NFL);
                        float er, ei, dr = 1.0f, di = 0.0f;
                        if (UNIFORM) {
                            phasor_f32(ph * fr.kf[c0], er, ei);
                            if (FT > 1) phasor_f32(ph * dkf, dr, di);
                        }
#pragma unroll
                        for (int c = 0; c < FT; c++) {
                            if (!UNIFORM) phasor_f32(ph * fr.kf[min(c0 + c, PRED_MAXF - 1)], er, ei);
                            if (!POL) {
                                const float f = fl[c];
                                fr_[c][0] = fmaf(f, er, fr_[c][0]);
                                fi_[c][0] = fmaf(f, ei, fi_[c][0]);
                            } else {
                                const float fa = fl[4 * c], fd = fl[4 * c + 1], fu = fl[4 * c + 2], fv = fl[4 * c + 3];
                                fr_[c][0] = fmaf(fa, er, fr_[c][0]);
                                fi_[c][0] = fmaf(fa, ei, fi_[c][0]);
                                fr_[c][3] = fmaf(fd, er, fr_[c][3]);
                                fi_[c][3] = fmaf(fd, ei, fi_[c][3]);
                                fr_[c][1] = fmaf(-fv, ei, fmaf(fu, er, fr_[c][1]));
                                fi_[c][1] = fmaf(fv, er, fmaf(fu, ei, fi_[c][1]));
                                fr_[c][2] = fmaf(fv, ei, fmaf(fu, er, fr_[c][2]));
                                fi_[c][2] = fmaf(-fv, er, fmaf(fu, ei, fi_[c][2]));
                            }
                            if (UNIFORM && c + 1 < FT) {
                                const float nr = fmaf(-ei, di, er * dr), ni = fmaf(ei, dr, er * di);
                                er = nr; ei = ni;
                            }
                        }
                    }
#pragma unroll
                    for (int c = 0; c < FT; c++)
#pragma unroll
                        for (int j = 0; j < NACC; j++) { acc[c][j].re += (double)fr_[c][j]; acc[c][j].im += (double)fi_[c][j]; }
                }
            } else {
#pragma unroll 2
            for (int s = 0; s < ns; s++) {
                const double ph = fma(w, s_n[s], fma(v, s_m[s], u * s_l[s]));  // metres
                const double* fl = s_fl + s * (FT * NFL);
                double er, ei, dr = 1.0, di = 0.0;
                double pr = 0.0, pi_ = 0.0, twodr = 2.0;
                if (UNIFORM) {
                    phasor_f64(ph * fr.kf[c0], s_tab, er, ei);
                    if (FT > 1) { phasor_f64(ph * dkf, s_tab, dr, di); twodr = dr + dr; }
                }
#pragma unroll
                for (int c = 0; c < FT; c++) {
                    if (!UNIFORM) phasor_f64(ph * fr.kf[min(c0 + c, PRED_MAXF - 1)], s_tab, er, ei);
                    if (!POL) {
                        const double f = fl[c];
                        acc[c][0].re = fma(f, er, acc[c][0].re);
                        acc[c][0].im = fma(f, ei, acc[c][0].im);
                    } else {
                        const double fa = fl[4 * c], fd = fl[4 * c + 1], fu = fl[4 * c + 2], fv = fl[4 * c + 3];
                        acc[c][0].re = fma(fa, er, acc[c][0].re);   // XX = (I+Q) e
                        acc[c][0].im = fma(fa, ei, acc[c][0].im);
                        acc[c][3].re = fma(fd, er, acc[c][3].re);   // YY = (I-Q) e
                        acc[c][3].im = fma(fd, ei, acc[c][3].im);
                        // XY = (U+iV) e,  YX = (U-iV) e,  e = er + i ei
                        acc[c][1].re = fma(-fv, ei, fma(fu, er, acc[c][1].re));
                        acc[c][1].im = fma(fv, er, fma(fu, ei, acc[c][1].im));
                        acc[c][2].re = fma(fv, ei, fma(fu, er, acc[c][2].re));
                        acc[c][2].im = fma(-fv, er, fma(fu, ei, acc[c][2].im));
                    }
                    if (UNIFORM && c + 1 < FT) {
                        // e_{c+1} = e_c d for the first step, then the three-term form e_{c+1} = 2 Re(d) e_c - e_{c-1}
                        // (exact for a geometric sequence of unit phasors; 2 instead of 4 instructions per channel)
                        double nr, ni;
                        if (c == 0) { nr = fma(-ei, di, er * dr); ni = fma(ei, dr, er * di); }
                        else { nr = fma(twodr, er, -pr); ni = fma(twodr, ei, -pi_); }
                        pr = er; pi_ = ei;
                        er = nr; ei = ni;
                    }
                }
            }
            }
        }
        if (live) {
            if (SCALAR) {
                sagecal_c128* o = coh + ((size_t)k * rows + r) * F + c0;
#pragma unroll
                for (int c = 0; c < FT; c++)
                    if (c0 + c < F) { o[c].re = acc[c][0].re; o[c].im = acc[c][0].im; }
            } else {
                sagecal_c128* o = coh + (((size_t)k * rows + r) * F + c0) * 4;
#pragma unroll
                for (int c = 0; c < FT; c++) {
                    if (c0 + c < F) {
                        if (!POL) {
                            stg256(o + 4 * c, acc[c][0].re, acc[c][0].im, 0.0, 0.0);
                            stg256(o + 4 * c + 2, 0.0, 0.0, acc[c][0].re, acc[c][0].im);
                        } else {
                            stg256(o + 4 * c, acc[c][0].re, acc[c][0].im, acc[c][1].re, acc[c][1].im);
                            stg256(o + 4 * c + 2, acc[c][2].re, acc[c][2].im, acc[c][3].re, acc[c][3].im);
                        }
                    }
                }
            }
            if (RESID) {
                // R -= J_p C J_q^H for this cluster: unpolarised C = c I2, so the model is c (J_p J_q^H)
                m22 jp, jq, pq;
                load_jones(rs.jones + ((size_t)k * rs.N + sp) * 4, jp);
                load_jones(rs.jones + ((size_t)k * rs.N + sq) * 4, jq);
                if (!POL) mmh(jp, jq, pq);
#pragma unroll
                for (int c = 0; c < FT; c++) {
                    if (c0 + c < F) {
                        m22 md;
                        if (!POL) {
#pragma unroll
                            for (int e = 0; e < 4; e++) md.a[e] = cmul(acc[c][0], pq.a[e]);
                        } else {
                            m22 cc, t1;
#pragma unroll
                            for (int e = 0; e < 4; e++) cc.a[e] = acc[c][POL ? e : 0];
                            mm(jp, cc, t1);
                            mmh(t1, jq, md);
                        }
#pragma unroll
                        for (int e = 0; e < 4; e++) {
                            double2 x = s_res[(4 * c + e) * PRED_THREADS];
                            x.x -= md.a[e].re; x.y -= md.a[e].im;
                            s_res[(4 * c + e) * PRED_THREADS] = x;
                        }
                    }
                }
            }
        }
      }
      if (RESID && live) {
#pragma unroll
          for (int c = 0; c < FT; c++) {
              if (c0 + c < F) {
                  sagecal_c128* ro = rs.residual + ((size_t)r * F + c0 + c) * 4;
                  const double2 a0 = s_res[(4 * c) * PRED_THREADS], a1 = s_res[(4 * c + 1) * PRED_THREADS];
                  const double2 a2 = s_res[(4 * c + 2) * PRED_THREADS], a3 = s_res[(4 * c + 3) * PRED_THREADS];
                  stg256(ro, a0.x, a0.y, a1.x, a1.y);
                  stg256(ro + 2, a2.x, a2.y, a3.x, a3.y);
              }
          }
      }
    }
}

// ---- unpolarised float64 prediction, RPT rows per thread ---------------------------------------------------------------
// The hot loop is held back by its shared-memory reads (profiles/r02_ncu_full_predict_cfg4.md): with RPT = 2 rows per
// thread a source's position and its FT fluxes are read once for both.  Rows r, r + 128, ... of an RPT x 128-row tile, so
// that a warp's uvw reads and coherency stores stay contiguous.  Same arithmetic per (row, source) as predict_kernel:
// bit-identical output.
template <int FT, bool UNIFORM, bool SCALAR, int RPT, int MINB>
__global__ void __launch_bounds__(PRED_THREADS, MINB)
predict2_kernel(int64_t rows, int F, int Fpad, PredFreqs fr, double dkf, PredClusters cl,
                const double* __restrict__ uvw, const double* __restrict__ src_l,
                const double* __restrict__ src_m, const double* __restrict__ nm1_g,
                const double* __restrict__ flux_g, sagecal_c128* __restrict__ coh) {
    constexpr int ST = 128;
    __shared__ double s_l[ST], s_m[ST], s_n[ST];
    __shared__ __align__(16) double s_fl[ST * FT];
    __shared__ double2 s_tab_all[64 * 8];
    if (threadIdx.x < 64) {
        double sn, cs;
        sincospi((double)threadIdx.x * 0.03125, &sn, &cs);
#pragma unroll
        for (int c = 0; c < 8; c++) s_tab_all[8 * threadIdx.x + c] = make_double2(cs, sn);
    }
    const unsigned s_tab = (unsigned)__cvta_generic_to_shared(s_tab_all + (threadIdx.x & 7));
    const int k = blockIdx.y;
    const int s_begin = cl.off[k], s_end = cl.off[k + 1];
    int64_t r[RPT];
    bool live[RPT];
    double u[RPT], v[RPT], w[RPT];
#pragma unroll
    for (int t = 0; t < RPT; t++) {
        r[t] = (int64_t)blockIdx.x * (RPT * PRED_THREADS) + t * PRED_THREADS + threadIdx.x;
        live[t] = r[t] < rows;
        u[t] = v[t] = w[t] = 0.0;
        if (live[t]) { u[t] = uvw[3 * r[t]]; v[t] = uvw[3 * r[t] + 1]; w[t] = uvw[3 * r[t] + 2]; }
    }
    for (int c0 = 0; c0 < Fpad; c0 += FT) {
        cplx acc[RPT][FT][1];
#pragma unroll
        for (int t = 0; t < RPT; t++)
#pragma unroll
            for (int c = 0; c < FT; c++) acc[t][c][0] = mk(0.0, 0.0);
        for (int sb = s_begin; sb < s_end; sb += ST) {
            const int ns = min(ST, s_end - sb);
            __syncthreads();
            for (int i = threadIdx.x; i < ns; i += PRED_THREADS) {
                s_l[i] = src_l[sb + i]; s_m[i] = src_m[sb + i]; s_n[i] = nm1_g[sb + i];
            }
            for (int i = threadIdx.x; i < ns * FT; i += PRED_THREADS) {
                const int s = i / FT, rem = i - s * FT;
                s_fl[i] = flux_g[(size_t)(sb + s) * Fpad + c0 + rem];
            }
            __syncthreads();
            for (int s = 0; s < ns; s++) {
                const double sl = s_l[s], smm = s_m[s], sn = s_n[s];
                double fl[FT];
#pragma unroll
                for (int c = 0; c < FT; c++) fl[c] = s_fl[s * FT + c];
#pragma unroll
                for (int t = 0; t < RPT; t++) {
                    const double ph = fma(w[t], sn, fma(v[t], smm, u[t] * sl));  // metres
                    double er, ei, dr = 1.0, di = 0.0;
                    double pr = 0.0, pi_ = 0.0, twodr = 2.0;
                    if (UNIFORM) {
                        phasor_f64(ph * fr.kf[c0], s_tab, er, ei);
                        if (FT > 1) { phasor_f64(ph * dkf, s_tab, dr, di); twodr = dr + dr; }
                    }
#pragma unroll
                    for (int c = 0; c < FT; c++) {
                        if (!UNIFORM) phasor_f64(ph * fr.kf[min(c0 + c, PRED_MAXF - 1)], s_tab, er, ei);
                        acc[t][c][0].re = fma(fl[c], er, acc[t][c][0].re);
                        acc[t][c][0].im = fma(fl[c], ei, acc[t][c][0].im);
                        if (UNIFORM && c + 1 < FT) {
                            double nr, ni;
                            if (c == 0) { nr = fma(-ei, di, er * dr); ni = fma(ei, dr, er * di); }
                            else { nr = fma(twodr, er, -pr); ni = fma(twodr, ei, -pi_); }
                            pr = er; pi_ = ei;
                            er = nr; ei = ni;
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int t = 0; t < RPT; t++) {
            if (!live[t]) continue;
            if (SCALAR) {
                sagecal_c128* o = coh + ((size_t)k * rows + r[t]) * F + c0;
#pragma unroll
                for (int c = 0; c < FT; c++)
                    if (c0 + c < F) { o[c].re = acc[t][c][0].re; o[c].im = acc[t][c][0].im; }
            } else {
                sagecal_c128* o = coh + (((size_t)k * rows + r[t]) * F + c0) * 4;
#pragma unroll
                for (int c = 0; c < FT; c++) {
                    if (c0 + c < F) {
                        stg256(o + 4 * c, acc[t][c][0].re, acc[t][c][0].im, 0.0, 0.0);
                        stg256(o + 4 * c + 2, 0.0, 0.0, acc[t][c][0].re, acc[t][c][0].im);
                    }
                }
            }
        }
    }
}

template <int FT, bool POL, bool UNIFORM, bool SCALAR, bool MIXED>
static int launch_predict(dim3 grid, cudaStream_t st, int64_t rows, int F, int Fpad, const PredFreqs& fr, double dkf,
                          const PredClusters& cl, const double* uvw, const double* l, const double* m,
                          const double* nm1, const double* flux, sagecal_c128* coh, const PredResid* rs) {
    LaunchScope ls(KK_PREDICT, st);
    if (rs) {
        if (MIXED) return SAGECAL_EUNSUPPORTED;
        // the residual tile: FT channels x 4 correlations x 16 B per thread (64 KB at FT = 8), opted in per device
        constexpr int smem = FT * 4 * PRED_THREADS * 16;
        auto kern = predict_kernel<FT, POL, UNIFORM, SCALAR, false, true>;
        static bool ready[64] = {};
        static std::mutex mu;                          // two host threads may meet here on their first call
        std::lock_guard<std::mutex> lk(mu);
        int dev = 0;
        SGC_CUDA(cudaGetDevice(&dev));
        if (dev < 0 || dev >= 64) return SAGECAL_EUNSUPPORTED;
        if (!ready[dev]) {
            SGC_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            ready[dev] = true;
        }
        kern<<<dim3(grid.x, 1), PRED_THREADS, smem, st>>>(rows, F, Fpad, fr, dkf, cl, uvw, l, m, nm1, flux, coh, *rs);
    } else if (!POL && !MIXED) {
        // two rows per thread at four CTAs per SM (127 registers, no spills): 28.8 ms at configs[4] against 31.4 for
        // one row per thread, 29.1 at three CTAs per SM, 30.2 with three rows per thread
        const dim3 g2((unsigned)((rows + PRED_RPT * PRED_THREADS - 1) / (PRED_RPT * PRED_THREADS)), grid.y);
        predict2_kernel<FT, UNIFORM, SCALAR, PRED_RPT, 4><<<g2, PRED_THREADS, 0, st>>>(rows, F, Fpad, fr, dkf, cl, uvw, l, m, nm1,
                                                                                  flux, coh);
    } else {
        predict_kernel<FT, POL, UNIFORM, SCALAR, MIXED, false><<<grid, PRED_THREADS, 0, st>>>(rows, F, Fpad, fr, dkf, cl, uvw,
                                                                                     l, m, nm1, flux, coh, PredResid{});
    }
    SGC_LAUNCH_CHECK();
    return SAGECAL_OK;
}

static int pick_ft(int F) { return F >= 8 ? 8 : F >= 4 ? 4 : F >= 2 ? 2 : 1; }

}  // namespace sgc

using namespace sgc;

extern "C" size_t sagecal_predict_workspace_bytes(int nchan, int nsrc_total) {
    if (nchan < 1 || nchan > PRED_MAXF || nsrc_total < 0) return 0;
    const int ft = pick_ft(nchan);
    const size_t Fpad = round_up((size_t)nchan, ft);
    // nm1[S] + flux[S][Fpad][4]
    return round_up(sizeof(double) * (size_t)nsrc_total, 256) + round_up(sizeof(double) * (size_t)nsrc_total * Fpad * 4, 256) + 256;
}

static int predict_impl(int N, int T, int F, const double* freqs_host, double f0,
                        const double* uvw, int K, const int* cluster_offset_host,
                        const double* src_l, const double* src_m, const double* src_I,
                        const double* src_Q, const double* src_U, const double* src_V,
                        const double* src_alpha, int coh_format, sagecal_c128* coh,
                        int precision, void* workspace, size_t workspace_bytes, void* stream, const PredResid* rs) {
    if (N < 2 || T < 1 || F < 1 || F > PRED_MAXF || K < 0 || K > PRED_MAXK) return SAGECAL_EINVAL;
    if (!freqs_host || !(f0 > 0.0) || !cluster_offset_host) return SAGECAL_EINVAL;
    if (coh_format != SAGECAL_COH_FULL && coh_format != SAGECAL_COH_SCALAR) return SAGECAL_EINVAL;
    if (precision != 0 && precision != 1) return SAGECAL_EINVAL;
    const bool pol = src_Q || src_U || src_V;
    if (pol && !(src_Q && src_U && src_V)) return SAGECAL_EINVAL;
    if (pol && coh_format == SAGECAL_COH_SCALAR) return SAGECAL_EINVAL;
    if (K == 0) return SAGECAL_OK;
    if (cluster_offset_host[0] != 0) return SAGECAL_EINVAL;
    for (int k = 0; k < K; k++)
        if (cluster_offset_host[k + 1] < cluster_offset_host[k]) return SAGECAL_EINVAL;
    const int S = cluster_offset_host[K];
    if (!uvw || !coh || !aligned(coh, 32) || !aligned(uvw, 8)) return SAGECAL_EINVAL;
    if (S > 0 && (!src_l || !src_m || !src_I || !src_alpha)) return SAGECAL_EINVAL;
    for (int c = 0; c < F; c++)
        if (!(freqs_host[c] > 0.0)) return SAGECAL_EINVAL;
    if (!workspace || !aligned(workspace, 256) || workspace_bytes < sagecal_predict_workspace_bytes(F, S))
        return SAGECAL_EWORKSPACE;

    cudaStream_t st = (cudaStream_t)stream;
    const int ft = pick_ft(F);
    const int Fpad = (int)round_up((size_t)F, ft);
    const int64_t rows = (int64_t)T * ((int64_t)N * (N - 1) / 2);

    PredFreqs fr;
    for (int c = 0; c < PRED_MAXF; c++) fr.kf[c] = 0.0;
    for (int c = 0; c < F; c++) fr.kf[c] = freqs_host[c] / SAGECAL_C0;
    // Uniform spacing enables the channel recurrence.  The tile's phasors advance by df, so a channel that is off the
    // even grid by e Hz is off in phase by ph e / c0 cycles (ph up to 1e4 m): the test admits a few ulp of the
    // frequency (4 eps f = 1.4e-7 Hz at 160 MHz, 5e-12 cycles), nothing a parity bound of 1e-10 could see.
    bool uniform = true;
    double df = F > 1 ? (freqs_host[F - 1] - freqs_host[0]) / (F - 1) : 0.0;
    for (int c = 0; c < F; c++)
        if (fabs(freqs_host[c] - (freqs_host[0] + c * df)) > 4.0 * 2.220446049250313e-16 * fabs(freqs_host[F - 1])) uniform = false;
    const double dkf = df / SAGECAL_C0;
    for (int c = F; c < Fpad; c++) fr.kf[c] = fr.kf[0] + c * dkf;  // padded channels: harmless phases, zero flux
    PredClusters cl;
    for (int k = 0; k <= PRED_MAXK; k++) cl.off[k] = cluster_offset_host[k <= K ? k : K];

    double* nm1 = (double*)workspace;
    double* flux = (double*)((char*)workspace + round_up(sizeof(double) * (size_t)S, 256));
    if (S > 0) {
        const int n = S * Fpad, tb = 256;
        LaunchScope ls(KK_PREP, st);
        if (pol)
            predict_prep_kernel<4><<<(n + tb - 1) / tb, tb, 0, st>>>(S, F, Fpad, fr, SAGECAL_C0 / f0, src_l, src_m, src_I,
                                                                   src_Q, src_U, src_V, src_alpha, nm1, flux);
        else
            predict_prep_kernel<1><<<(n + tb - 1) / tb, tb, 0, st>>>(S, F, Fpad, fr, SAGECAL_C0 / f0, src_l, src_m, src_I,
                                                                   nullptr, nullptr, nullptr, src_alpha, nm1, flux);
        SGC_LAUNCH_CHECK();
    }
    dim3 grid((unsigned)((rows + PRED_THREADS - 1) / PRED_THREADS), (unsigned)K);
    const bool scalar = coh_format == SAGECAL_COH_SCALAR;
    const bool mixed = precision == 1;
#define SGC_PRED(FT_, POL_, UNI_, SC_)                                                                                  \
    do {                                                                                                               \
        if (mixed) return launch_predict<FT_, POL_, UNI_, SC_, true>(grid, st, rows, F, Fpad, fr, dkf, cl, uvw, src_l,  \
                                                                    src_m, nm1, flux, coh, rs);                        \
        return launch_predict<FT_, POL_, UNI_, SC_, false>(grid, st, rows, F, Fpad, fr, dkf, cl, uvw, src_l, src_m,    \
                                                          nm1, flux, coh, rs);                                         \
    } while (0)
#define SGC_PRED_FT(FT_)                                            \
    do {                                                            \
        if (pol) { if (uniform) SGC_PRED(FT_, true, true, false); else SGC_PRED(FT_, true, false, false); } \
        else if (scalar) { if (uniform) SGC_PRED(FT_, false, true, true); else SGC_PRED(FT_, false, false, true); } \
        else { if (uniform) SGC_PRED(FT_, false, true, false); else SGC_PRED(FT_, false, false, false); } \
    } while (0)
    switch (ft) {
        case 8: SGC_PRED_FT(8); break;
        case 4: SGC_PRED_FT(4); break;
        case 2: SGC_PRED_FT(2); break;
        default: SGC_PRED_FT(1); break;
    }
#undef SGC_PRED_FT
#undef SGC_PRED
    return SAGECAL_OK;
}

extern "C" int sagecal_predict_coherencies(int N, int T, int F, const double* freqs_host, double f0,
                                           const double* uvw, int K, const int* cluster_offset_host,
                                           const double* src_l, const double* src_m, const double* src_I,
                                           const double* src_Q, const double* src_U, const double* src_V,
                                           const double* src_alpha, int coh_format, sagecal_c128* coh,
                                           int precision, void* workspace, size_t workspace_bytes, void* stream) {
    return predict_impl(N, T, F, freqs_host, f0, uvw, K, cluster_offset_host, src_l, src_m, src_I, src_Q, src_U, src_V,
                        src_alpha, coh_format, coh, precision, workspace, workspace_bytes, stream, nullptr);
}

// ---- no-allocation entry point (README "Callers that cannot allocate") ------------------------------------------------
// Same prediction as sagecal_predict_coherencies, with the prepared source table (nm1[S], flux[S][Fpad][NFL]: what
// predict_prep_kernel writes and the predict kernels read) in a file-scope device array instead of a caller's
// workspace.  Every device that loads the library holds SAGECAL_PREDICT_STATIC_BYTES of it until the process exits.
// The name `g_predict_scratch` is only a stand-in in host code: the device address comes from cudaGetSymbolAddress, once
// per device, with that device current.
static __device__ __align__(256) unsigned char g_predict_scratch[SAGECAL_PREDICT_STATIC_BYTES];

static int predict_static_scratch(void** out) {
    static void* addr[64] = {};
    static std::mutex mu;                              // two host threads may meet here on their first call
    std::lock_guard<std::mutex> lk(mu);
    int dev = 0;
    SGC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return SAGECAL_EUNSUPPORTED;
    if (!addr[dev]) {
        void* ptr = nullptr;
        SGC_CUDA(cudaGetSymbolAddress(&ptr, g_predict_scratch));
        if (!ptr || !aligned(ptr, 256)) return SAGECAL_EUNSUPPORTED;
        addr[dev] = ptr;
    }
    *out = addr[dev];
    return SAGECAL_OK;
}

extern "C" size_t sagecal_predict_static_bytes(void) { return (size_t)SAGECAL_PREDICT_STATIC_BYTES; }

extern "C" int sagecal_predict_coherencies_static(int N, int T, int F, const double* freqs_host, double f0,
                                                  const double* uvw, int K, const int* cluster_offset_host,
                                                  const double* src_l, const double* src_m, const double* src_I,
                                                  const double* src_Q, const double* src_U, const double* src_V,
                                                  const double* src_alpha, int coh_format, sagecal_c128* coh,
                                                  int precision, void* stream) {
    if (F < 1 || F > PRED_MAXF || K < 0 || K > PRED_MAXK || !cluster_offset_host) return SAGECAL_EINVAL;
    const int S = cluster_offset_host[K];
    if (S < 0) return SAGECAL_EINVAL;
    // the source table must fit the fixed array: nothing is allocated here, so a larger sky model is refused
    const size_t need = sagecal_predict_workspace_bytes(F, S);
    if (need == 0 || need > (size_t)SAGECAL_PREDICT_STATIC_BYTES) return SAGECAL_ESTATICLIMIT;
    void* scratch = nullptr;
    int rc;
    if ((rc = predict_static_scratch(&scratch))) return rc;
    // predict_prep_kernel writes every entry of the table the predict kernel reads: nothing has to start at zero
    return predict_impl(N, T, F, freqs_host, f0, uvw, K, cluster_offset_host, src_l, src_m, src_I, src_Q, src_U, src_V,
                        src_alpha, coh_format, coh, precision, scratch, (size_t)SAGECAL_PREDICT_STATIC_BYTES, stream, nullptr);
}

extern "C" int sagecal_predict_residual(int N, int T, int F, const double* freqs_host, double f0,
                                        const double* uvw, int K, const int* cluster_offset_host,
                                        const double* src_l, const double* src_m, const double* src_I,
                                        const double* src_Q, const double* src_U, const double* src_V,
                                        const double* src_alpha, int coh_format, sagecal_c128* coh,
                                        const sagecal_c128* jones, const sagecal_c128* vis, sagecal_c128* residual,
                                        void* workspace, size_t workspace_bytes, void* stream) {
    if (N < 2 || T < 1 || F < 1 || K < 1) return SAGECAL_EINVAL;
    if (!jones || !vis || !residual || !aligned(jones, 16) || !aligned(vis, 32) || !aligned(residual, 32)) return SAGECAL_EINVAL;
    PredResid rs;
    rs.N = N; rs.K = K; rs.B = (int64_t)N * (N - 1) / 2;
    rs.jones = jones; rs.vis = vis; rs.residual = residual;
    return predict_impl(N, T, F, freqs_host, f0, uvw, K, cluster_offset_host, src_l, src_m, src_I, src_Q, src_U, src_V,
                        src_alpha, coh_format, coh, 0, workspace, workspace_bytes, stream, &rs);
}
