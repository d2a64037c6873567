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
// sagecal_predict_set_form: 0 = station form when the uvw allow it (default), 1 = always one phasor per (baseline, source)
static int g_predict_form = 0;
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
                const double* __restrict__ flux_g, sagecal_c128* __restrict__ coh,
                const int* __restrict__ only_if_flag) {
    // launched behind predict_station_kernel: runs only if the uvw were found not to be station differences
    if (only_if_flag && *only_if_flag == 0) return;
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

// ---- unpolarised float64 prediction in STATION form: a dense contraction on the FP64 tensor cores -------------------
// An interferometer's uvw are differences of station coordinates: u_pq = x_q - x_p with x_s = u_0s (the rows of the
// baselines (0, s); x_0 = 0), whichever sign convention the caller's uvw follow.  Then
//     exp(-2 pi i kappa (x_q - x_p).s) = e_q,s conj(e_p,s),   e_p,s = exp(-2 pi i kappa x_p.s)
//     C_pq[c] = sum_s conj(e_p,s[c]) (f_s[c] e_q,s[c])
// i.e. per (time slot, cluster, channel) a rank-S_k Hermitian update -- 4 real FMAs per (visibility, source) instead of
// the 8.8 FP64 instructions of a phasor per (baseline, source), and N S phasors per time slot instead of B S.  In real
// form C = A B with A = [Re e_p | Im e_p] (stations x 2 S_k) for the real and A' = [-Im e_p | Re e_p] for the imaginary
// part, B = [Re f e_q ; Im f e_q]: DMMA m8n8k4, one k-step = two sources.
//
// station_phasor_kernel writes the phasors once per (time slot, station, source) -- E = e and FE = f e, as
// [t][source pair][channel][station][2 sources x (re, im)] -- into the part of the workspace beyond
// sagecal_predict_workspace_bytes() (the time slots are predicted in chunks of what fits there).
// predict_station_kernel: a CTA takes a 16 x 32 tile of station pairs (p-tile <= q-tile) of one time slot and every
// PG_KZ-th cluster.  Eight warps; a warp contracts ONE channel x 16 p x 32 q: 2 x 4 blocks of m8n8k4 x {Re, Im} = 32
// accumulator doubles per lane (two CTAs = 16 warps per SM).  The operand rows (512 B of the p stations from E, 1 KB of
// the q stations from FE per (pair, channel)) arrive by cp.async in a multi-stage pipeline, laid out so that every
// fragment load is conflict-free; per k-step a warp issues 8 LDS.64 -- A for two m-tiles, A' = the partner entry with
// its sign bit flipped, B for four n-tiles -- for 16 DMMAs.  Blocks entirely at or below the diagonal do no
// arithmetic.  A DMMA holds its scheduler's issue port for the 16 cycles it occupies the pipe, so every other
// instruction costs its cycle in full: the copy addresses are fixed per thread and advance by increments.
// The finished tile goes through shared memory as [c][p][q] and leaves in the order of global memory (consecutive
// threads store consecutive 32-byte pieces: whole lines); with 2x2 output it has a buffer of its own and leaves row by
// row during the NEXT tile's contraction (PgCfg below).  profiles/r02_ncu_predict_station.md has the measurements.
//
// uvw_station_check_kernel decides on the device whether the caller's uvw ARE station-consistent (every row within
// 8 eps of u_0q - u_0p, relative to the 1-norms of the three vectors: rounding, nothing a parity bound of 1e-10 sees
// since the phase error is 2 pi kappa |d| |s| < 1e-11 rad for 20 km baselines and a 5 degree field); if
// not, this kernel returns at once and predict2_kernel (launched after it, told to return in the other case) does the
// work: no host synchronisation either way.
constexpr int PG_TP = 16, PG_TQ = 32;   // CTA tile: 16 row stations x 32 column stations
#ifndef PG_KZ_
#define PG_KZ_ 5
#endif
#ifndef PG_KSS_
#define PG_KSS_ 2
#endif
#ifndef PG_NSTG_
#define PG_NSTG_ 4
#endif
constexpr int PG_KZ = PG_KZ_;                // the clusters are dealt to this many CTAs per (tile, time slot)
constexpr int PG_KSS = PG_KSS_;               // k-steps (source pairs) per pipeline stage
constexpr int PG_NSTG = PG_NSTG_;              // stages in flight
constexpr int PG_THREADS = 256;
struct PredPairs { int off[PRED_MAXK + 1]; };            // first source PAIR of every cluster (a cluster with an odd
                                                         // count ends in a padding source of zero flux)
// 2x2 output: the finished tile has a shared-memory buffer of its own and leaves row by row while the NEXT tile is
// contracted (one stage = one source pair, three in flight: what fits next to the 68 KB tile at two CTAs per SM);
// scalar output (a quarter of the bytes, whose stores cost nothing) keeps the larger stages and sends the tile out at
// once through the operand buffers.  configs[4]: 17.8 against 19.6 ms (2x2), 14.7 against 15.7 ms (scalar).
template <bool SCALAR> struct PgCfg {
    static constexpr bool PIPE = !SCALAR;
    static constexpr int KSS = PIPE ? 1 : PG_KSS;        // k-steps (source pairs) per pipeline stage
    static constexpr int NSTG = PIPE ? 3 : PG_NSTG;      // stages in flight
};
template <int FT, bool SCALAR> constexpr size_t pg_smem_bytes() {
    constexpr size_t stages = sizeof(double) * (size_t)(PgCfg<SCALAR>::NSTG * PgCfg<SCALAR>::KSS * FT * (PG_TP + PG_TQ) * 4);
    constexpr size_t tile = sizeof(double) * 2 * (size_t)FT * (PG_TP * (PG_TQ + 1) + 1);
    return PgCfg<SCALAR>::PIPE ? stages + tile : (stages > tile ? stages : tile);
}
// bytes of station phasors (both operands) per time slot
static size_t pg_bytes_per_slot(int N, int npairs, int Fpad) { return (size_t)2 * npairs * Fpad * N * 4 * sizeof(double); }
// tiles of one time slot: p-tile pi meets the q-tiles from the one that holds its first station on
static int64_t pg_tiles(int N) {
    const int ntp = (N + PG_TP - 1) / PG_TP, ntq = (N + PG_TQ - 1) / PG_TQ;
    int64_t n = 0;
    for (int pi = 0; pi < ntp; pi++) n += ntq - (pi * PG_TP) / PG_TQ;
    return n;
}
__device__ __forceinline__ void pg_cp_async16(void* smem, const void* gmem) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void pg_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_> __device__ __forceinline__ void pg_cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N_) : "memory"); }

// Station phasors of nt time slots from t0: E[t][pair][c][station][2 sources x (re, im)] = e_p,s[c] and FE = f_s[c] e.
// One thread per (t, pair, station, source of the pair), all FT-channel tiles; adjacent lanes write adjacent 16 bytes.
template <int FT, bool UNIFORM>
__global__ void __launch_bounds__(128)
station_phasor_kernel(int N, int64_t B, int F, int Fpad, int K, int npairs, int t0, PredFreqs fr, double dkf, PredClusters cl,
                      PredPairs pp, const double* __restrict__ uvw, const double* __restrict__ src_l,
                      const double* __restrict__ src_m, const double* __restrict__ nm1_g,
                      const double* __restrict__ flux_g, double* __restrict__ E, double* __restrict__ FE,
                      const int* __restrict__ flag) {
    if (*flag) return;
    __shared__ double2 s_tab_all[64 * 8];
    if (threadIdx.x < 64) {
        double sn, cs;
        sincospi((double)threadIdx.x * 0.03125, &sn, &cs);
#pragma unroll
        for (int c = 0; c < 8; c++) s_tab_all[8 * threadIdx.x + c] = make_double2(cs, sn);
    }
    __syncthreads();
    const unsigned s_tab = (unsigned)__cvta_generic_to_shared(s_tab_all + (threadIdx.x & 7));
    const int e = blockIdx.x * 128 + threadIdx.x;        // (station, h) within the pair
    const int pair = blockIdx.y, tl = blockIdx.z;
    if (e >= 2 * N) return;
    const int st = e >> 1, h = e & 1;
    // the pair's cluster: the last k with pp.off[k] <= pair
    int lo = 0, hi = K;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (pp.off[mid] <= pair) lo = mid; else hi = mid; }
    const int s = cl.off[lo] + 2 * (pair - pp.off[lo]) + h;
    const bool live = s < cl.off[lo + 1];                // else the padding source of an odd cluster
    double u = 0.0, v = 0.0, w = 0.0;
    if (st >= 1) {
        const double* x = uvw + 3 * ((int64_t)(t0 + tl) * B + (st - 1));      // x_s = u_0s, x_0 = 0
        u = x[0]; v = x[1]; w = x[2];
    }
    const double ph = live ? fma(w, nm1_g[s], fma(v, src_m[s], u * src_l[s])) : 0.0;   // metres
    for (int c0 = 0; c0 < Fpad; c0 += FT) {
        double er, ei, dr = 1.0, di = 0.0;
        double pr = 0.0, pi_ = 0.0, twodr = 2.0;
        if (UNIFORM) {
            phasor_f64(ph * fr.kf[c0], s_tab, er, ei);
            if (FT > 1) { phasor_f64(ph * dkf, s_tab, dr, di); twodr = dr + dr; }
        }
#pragma unroll
        for (int c = 0; c < FT; c++) {
            if (!UNIFORM) phasor_f64(ph * fr.kf[min(c0 + c, PRED_MAXF - 1)], s_tab, er, ei);
            const double f = live ? flux_g[(size_t)s * Fpad + c0 + c] : 0.0;
            const size_t o = ((((size_t)tl * npairs + pair) * Fpad + c0 + c) * N + st) * 4 + 2 * h;
            *reinterpret_cast<double2*>(E + o) = make_double2(er, ei);
            *reinterpret_cast<double2*>(FE + o) = make_double2(f * er, f * ei);
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

__global__ void uvw_station_check_kernel(int N, int64_t B, int64_t rows, const double* __restrict__ uvw, int* flag) {
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= rows) return;
    const int64_t t = r / B;
    int p, q;
    bl_stations(N, r - t * B, p, q);
    if (p == 0) return;                                  // these rows DEFINE the station coordinates
    const double* x = uvw + 3 * r;
    const double* a = uvw + 3 * (t * B + (p - 1));       // bl_index(N, 0, s) = s - 1
    const double* c = uvw + 3 * (t * B + (q - 1));
    // uvw components are sums of products of coordinates that may cancel: the rounding of a component scales with the
    // vectors' size, not with its own (measured on the generator's tracks: up to 1.25 eps of the 1-norms below)
    double scale = 0.0;
#pragma unroll
    for (int d = 0; d < 3; d++) scale += fabs(x[d]) + fabs(c[d]) + fabs(a[d]);
    const double tol = 8.0 * 2.220446049250313e-16 * scale;
    bool bad = false;
#pragma unroll
    for (int d = 0; d < 3; d++)
        if (!(fabs(x[d] - (c[d] - a[d])) <= tol)) bad = true;     // NaN is inconsistent
    if (bad) *flag = 1;                                  // every writer stores the same value
}

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <int FT, bool SCALAR>
__global__ void __launch_bounds__(PG_THREADS, 2)
predict_station_kernel(int N, int64_t B, int64_t rows, int F, int Fpad, int K, int npairs, int t0, PredPairs pp,
                       const double* __restrict__ E, const double* __restrict__ FE, sagecal_c128* __restrict__ coh,
                       const int* __restrict__ flag) {
    if (*flag) return;                                   // uvw are not station differences: predict2_kernel's job
    extern __shared__ __align__(16) unsigned char pg_smem[];
    constexpr bool PIPE = PgCfg<SCALAR>::PIPE;
    constexpr int KSS = PgCfg<SCALAR>::KSS, NSTG = PgCfg<SCALAR>::NSTG;
    constexpr int SZA = KSS * FT * PG_TP * 4;            // doubles per stage: [ks][c][station][2 sources x (re, im)]
    constexpr int SZB = KSS * FT * PG_TQ * 4;
    constexpr int SZS = SZA + SZB;
    // a warp takes ONE channel, all 16 p and NT n-tiles of 8 q (8 fragment loads per 16 DMMAs at FT = 8, 32
    // accumulator doubles per lane: 16 warps per SM)
    constexpr int NQW = 8 / FT < 4 ? 8 / FT : 4, NT = 4 / NQW;
    double* smem = reinterpret_cast<double*>(pg_smem);
    double2* s_stage = reinterpret_cast<double2*>(pg_smem) + (PIPE ? (NSTG * SZS) / 2 : 0);   // the finished tile: [c][p][q], padded
    // tile (pi, qi) of this CTA: p-tiles of PG_TP stations, q-tiles of PG_TQ; only tiles with some q > p
    const int ntq = (N + PG_TQ - 1) / PG_TQ;
    int pi = 0, rem = (int)blockIdx.x;
    while (rem >= ntq - (pi * PG_TP) / PG_TQ) { rem -= ntq - (pi * PG_TP) / PG_TQ; pi++; }
    const int qi = (pi * PG_TP) / PG_TQ + rem;
    const int p0 = PG_TP * pi, q0 = PG_TQ * qi;
    const int tl = blockIdx.y, t = t0 + tl;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, j = lane & 3;
    const int cw = warp % FT, qw = warp / FT;            // channel, q group of this warp
    const bool w_work = qw < NQW;                        // FT = 1: four of the eight warps contract
    const int qb = qw * (NT * 8);                        // first q of the warp within the tile
    unsigned act = 0;                                    // (m-tile, n-tile) blocks with some q > p (bit mt * NT + nt)
    if (w_work) {
#pragma unroll
        for (int mt = 0; mt < 2; mt++)
#pragma unroll
            for (int nt = 0; nt < NT; nt++)
                if (q0 + qb + nt * 8 + 7 > p0 + mt * 8 && p0 + mt * 8 < N && q0 + qb + nt * 8 < N) act |= 1u << (mt * NT + nt);
    }
    const bool all_act = act == (1u << (2 * NT)) - 1u;
    const int a_off = (cw * PG_TP + g) * 4 + j;
    const int b_off = SZA + (cw * PG_TQ + qb + g) * 4 + j;
    const int jx = (j ^ 1) - j;                          // the partner entry (s, 1 - ri) of this lane's (s, ri)
    const int sgn = (j & 1) ? 0 : (int)0x80000000;       // Im part: A'[(s, 0)] = -Im e, A'[(s, 1)] = +Re e

    // operand copies: threads 0..191 copy two (pair, channel) rows per pass, 96 16-byte pieces each (32 of the p
    // stations from E, 64 of the q stations from FE); everything that does not depend on the stage is fixed here
    const bool cp_thread = threadIdx.x < 192;
    const int cp_rp = threadIdx.x >= 96 ? 1 : 0, cp_u = threadIdx.x - 96 * cp_rp;
    const bool cp_p = cp_u < 2 * PG_TP;
    const int cp_st = cp_p ? cp_u >> 1 : (cp_u - 2 * PG_TP) >> 1;
    const double* cp_src = (cp_p ? E + (size_t)min(p0 + cp_st, N - 1) * 4 : FE + (size_t)min(q0 + cp_st, N - 1) * 4) + 2 * (cp_u & 1);
    const int cp_dst = (cp_p ? 0 : SZA) + cp_st * 4 + 2 * (cp_u & 1);
    const int cp_rstride = (cp_p ? PG_TP : PG_TQ) * 4;
    const size_t rowlen = (size_t)N * 4;                 // doubles per (pair, channel) row

    // the finished tile leaves while the NEXT tile is contracted: one row of it per pipeline stage
    constexpr int PSTR = PG_TQ + 1, CSTR = PG_TP * PSTR + 1;         // strides in complex numbers
    constexpr int PCS = SCALAR ? FT : 2 * FT;        // pieces per (p, q): 16 bytes per channel / 32 bytes per half
    constexpr int QPT = PG_THREADS / PCS;            // q's covered by the CTA per trip
    constexpr int RC = SCALAR ? 1 : 4;               // complex numbers per (row, channel)
    const int pc = threadIdx.x % PCS, qoff = threadIdx.x / PCS;
    const int so_c = SCALAR ? pc : pc >> 1;
    const double2* so_sc = s_stage + so_c * CSTR + qoff;
    const size_t rowc = (size_t)F * RC;              // complex numbers per row
    const int pend = min(PG_TP, N - 1 - p0);         // rows p >= N - 1 have no baseline
    int so_pl = 0, so_pend = 0;
    bool so_ok = false;
    sagecal_c128* so_o = coh;
    int so_q[(PG_TQ + QPT - 1) / QPT];               // this thread's q's (-1: outside the tile or the array)
#pragma unroll
    for (int x = 0; x < (PG_TQ + QPT - 1) / QPT; x++) {
        const int q = q0 + qoff + x * QPT;
        so_q[x] = (qoff + x * QPT < PG_TQ && q < N) ? q : -1;
    }
    auto stream_row = [&]() {
        if (so_pl < so_pend) {
            const int p = p0 + so_pl;
#pragma unroll
            for (int x = 0; x < (PG_TQ + QPT - 1) / QPT; x++) {
                if (p < so_q[x] && so_ok) {
                    const double2 v = so_sc[so_pl * PSTR + x * QPT];
                    sagecal_c128* ox = so_o + (size_t)(x * QPT) * rowc;
                    if (SCALAR) *reinterpret_cast<double2*>(ox) = v;
                    else if (pc & 1) stg256(ox, 0.0, 0.0, v.x, v.y);
                    else stg256(ox, v.x, v.y, 0.0, 0.0);
                }
            }
            so_o += (size_t)(N - p - 2) * rowc;
            so_pl++;
        }
    };

    for (int k = blockIdx.z; k < K; k += gridDim.z) {
      const int pb = pp.off[k], np = pp.off[k + 1] - pb;
      const int nstage = (np + KSS - 1) / KSS;
      for (int c0 = 0; c0 < Fpad; c0 += FT) {
        double acc[2][NT][4];                            // [m-tile][n-tile][Re q, Re q+1, Im q, Im q+1]
#pragma unroll
        for (int mt = 0; mt < 2; mt++)
#pragma unroll
            for (int nt = 0; nt < NT; nt++)
#pragma unroll
                for (int x = 0; x < 4; x++) acc[mt][nt][x] = 0.0;

        // stage sg of this (cluster, channel tile): pairs pb + sg KSS ..; 16-byte pieces, 96 per (pair, channel)
        // running state of the copies: the next stage to issue, its buffer and its first row in global memory
        int isg = 0, ibuf = 0;
        const double* isrc = cp_src + (((size_t)tl * npairs + pb) * Fpad + c0 + (FT > 1 ? cp_rp : 0)) * rowlen;
        const size_t stage_rows = (size_t)KSS * Fpad * rowlen;
        auto issue = [&]() {
            if (isg < nstage && cp_thread) {
                // one pair per stage: running buffer index and pointer (fewer instructions between the DMMAs); the
                // two-pair stages of scalar output are faster with both recomputed (measured: 14.7 against 15.2 ms)
                double* dstg = smem + (KSS == 1 ? ibuf : isg % NSTG) * SZS + cp_dst;
                const int nrow = KSS == 1 ? FT : min(KSS, np - isg * KSS) * FT;
                const double* src = KSS == 1 ? isrc
                                             : cp_src + (((size_t)tl * npairs + pb + isg * KSS) * Fpad + c0 + (FT > 1 ? cp_rp : 0)) * rowlen;
                if (FT > 1) {
#pragma unroll
                    for (int ks = 0; ks < KSS; ks++) {
#pragma unroll
                        for (int c2 = 0; c2 < FT / 2; c2++) {
                            const int r = ks * FT + 2 * c2 + cp_rp;
                            if (KSS == 1 || r < nrow) pg_cp_async16(dstg + r * cp_rstride, src + c2 * (2 * rowlen));
                        }
                        src += Fpad * rowlen;
                    }
                } else {
#pragma unroll
                    for (int r0 = 0; r0 < KSS; r0 += 2) {
                        const int r = r0 + cp_rp;
                        if (r < nrow && r < KSS) pg_cp_async16(dstg + r * cp_rstride, src + (size_t)r * Fpad * rowlen);
                    }
                }
            }
            pg_cp_async_commit();                        // always: the group count per stage stays uniform
            isg++;
            isrc += stage_rows;
            ibuf = ibuf + 1 == NSTG ? 0 : ibuf + 1;
        };
        __syncthreads();                                 // every warp is done with the shared memory of the previous tile
#pragma unroll
        for (int sg = 0; sg < NSTG - 1; sg++) issue();
        int cbuf = 0;
        for (int sg = 0; sg < nstage; sg++) {
            pg_cp_async_wait<NSTG - 2>();             // stage sg has landed (this thread's part)
            __syncthreads();                             // ... everyone's; and stage sg - 1 has been consumed
            issue();
            const double* sb_ = smem + (KSS == 1 ? cbuf : sg % NSTG) * SZS;
            cbuf = cbuf + 1 == NSTG ? 0 : cbuf + 1;
            if (act) {
                const int nk = min(KSS, np - sg * KSS);
#pragma unroll
                for (int ks = 0; ks < KSS; ks++) {
                    if (ks > 0 && ks >= nk) break;       // only a cluster's last stage can be short
                    const double* ak = sb_ + a_off + ks * FT * PG_TP * 4;
                    const double* bk = sb_ + b_off + ks * FT * PG_TQ * 4;
                    double a[2], a2[2], b[NT];
#pragma unroll
                    for (int mt = 0; mt < 2; mt++) {
                        a[mt] = ak[mt * 32];
                        const double x = ak[mt * 32 + jx];
                        a2[mt] = __hiloint2double(__double2hiint(x) ^ sgn, __double2loint(x));
                    }
#pragma unroll
                    for (int nt = 0; nt < NT; nt++) b[nt] = bk[nt * 32];
                    if (all_act) {                       // every tile off the diagonal: no predicates in the way
#pragma unroll
                        for (int mt = 0; mt < 2; mt++)
#pragma unroll
                            for (int nt = 0; nt < NT; nt++) {
                                dmma884(acc[mt][nt][0], acc[mt][nt][1], a[mt], b[nt]);
                                dmma884(acc[mt][nt][2], acc[mt][nt][3], a2[mt], b[nt]);
                            }
                    } else {
#pragma unroll
                        for (int mt = 0; mt < 2; mt++)
#pragma unroll
                            for (int nt = 0; nt < NT; nt++)
                                if (act & (1u << (mt * NT + nt))) {
                                    dmma884(acc[mt][nt][0], acc[mt][nt][1], a[mt], b[nt]);
                                    dmma884(acc[mt][nt][2], acc[mt][nt][3], a2[mt], b[nt]);
                                }
                    }
                }
            }
            if (PIPE) stream_row();                      // a row of the previous tile
        }
        // the tile goes to shared memory as [c][p][q] complex, padded so that neither side has bank conflicts, and
        // leaves in the order of global memory: consecutive threads store consecutive 32-byte pieces (2x2 format: (v, 0)
        // and (0, v) of a (row, channel)) -- whole lines, 8 wavefronts per store instruction where lane-owns-its-rows
        // stores need 32
        if (PIPE) while (so_pl < so_pend) stream_row();  // what the stages did not cover
        __syncthreads();                                 // PIPE: the previous tile has been read; else: the last stage consumed
        if (w_work) {
#pragma unroll
            for (int mt = 0; mt < 2; mt++)
#pragma unroll
                for (int nt = 0; nt < NT; nt++)
#pragma unroll
                    for (int b = 0; b < 2; b++)
                        s_stage[cw * CSTR + (mt * 8 + g) * PSTR + qb + nt * 8 + 2 * j + b] = make_double2(acc[mt][nt][b], acc[mt][nt][2 + b]);
        }
        {   // this tile leaves during the next one (the next tile's first barrier orders these stores before the reads)
            const int inner = SCALAR ? (c0 + so_c) : (c0 + so_c) * 4 + 2 * (pc & 1);     // complex numbers into a row
            const int64_t row = (int64_t)t * B + row_start(N, p0) - p0 - 1 + q0 + qoff;
            so_o = coh + ((size_t)k * rows + (size_t)row) * rowc + inner;
            so_ok = c0 + so_c < F;
            so_pl = 0; so_pend = pend;
        }
        if (!PIPE) {                                     // the tile sits in the operand buffers: it leaves now
            __syncthreads();
            while (so_pl < so_pend) stream_row();
        }
      }
    }
    if (PIPE) {
        __syncthreads();
        while (so_pl < so_pend) stream_row();
    }
}

template <int FT, bool POL, bool UNIFORM, bool SCALAR, bool MIXED>
static int launch_predict(dim3 grid, cudaStream_t st, int64_t rows, int F, int Fpad, const PredFreqs& fr, double dkf,
                          const PredClusters& cl, const double* uvw, const double* l, const double* m,
                          const double* nm1, const double* flux, sagecal_c128* coh, const PredResid* rs, int N, int T,
                          int* flag, void* extra, size_t extra_bytes) {
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
        const int64_t B = (int64_t)N * (N - 1) / 2;
        const int64_t ntile = pg_tiles(N);
        const int K = (int)grid.y;
        // source pairs: a k-step of the contraction is two sources; a cluster with an odd count is padded
        PredPairs pp;
        int npairs = 0;
        for (int k = 0; k <= PRED_MAXK; k++) {
            pp.off[k] = npairs;
            if (k < K) npairs += (cl.off[k + 1] - cl.off[k] + 1) / 2;
        }
        const size_t per_slot = pg_bytes_per_slot(N, npairs, Fpad);
        const int64_t tchunk = per_slot ? (int64_t)(extra_bytes / per_slot) : 0;
        const bool station_form = g_predict_form == 0 && extra && tchunk >= 1 && npairs >= 1 && npairs <= 65535 &&
                                  ntile <= 0x7fffffff && 2 * (int64_t)N <= 0x7fffffff;
        if (station_form) {
            // station form first (returns at once if the uvw are not station differences), the per-baseline form behind
            // it (returns at once if they are): the choice is made on the device, nothing waits for the host
            constexpr int smem = (int)pg_smem_bytes<FT, SCALAR>();
            auto kern = predict_station_kernel<FT, SCALAR>;
            {
                static bool ready[64] = {};
                static std::mutex mu;                  // two host threads may meet here on their first call
                std::lock_guard<std::mutex> lk(mu);
                int dev = 0;
                SGC_CUDA(cudaGetDevice(&dev));
                if (dev < 0 || dev >= 64) return SAGECAL_EUNSUPPORTED;
                if (!ready[dev]) {
                    SGC_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
                    SGC_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
                    ready[dev] = true;
                }
            }
            SGC_CUDA(cudaMemsetAsync(flag, 0, sizeof(int), st));
            uvw_station_check_kernel<<<(unsigned)((rows + 255) / 256), 256, 0, st>>>(N, B, rows, uvw, flag);
            const int kz = K < PG_KZ ? K : PG_KZ;      // a CTA keeps its tile for several clusters
            const int tstep = (int)(tchunk < 32768 ? tchunk : 32768);
            count_more_launches(KK_PREDICT, 1 + 2 * ((T + tstep - 1) / tstep));     // the check, (phasors, contraction) per chunk
            for (int t0 = 0; t0 < T; t0 += tstep) {
                const int nt = T - t0 < tstep ? T - t0 : tstep;
                double* E = (double*)extra;
                double* FE = E + (size_t)nt * npairs * Fpad * N * 4;
                station_phasor_kernel<FT, UNIFORM><<<dim3((unsigned)((2 * N + 127) / 128), (unsigned)npairs, (unsigned)nt), 128, 0, st>>>(
                    N, B, F, Fpad, K, npairs, t0, fr, dkf, cl, pp, uvw, l, m, nm1, flux, E, FE, flag);
                kern<<<dim3((unsigned)ntile, (unsigned)nt, (unsigned)kz), PG_THREADS, smem, st>>>(
                    N, B, rows, F, Fpad, K, npairs, t0, pp, E, FE, coh, flag);
            }
        }
        predict2_kernel<FT, UNIFORM, SCALAR, PRED_RPT, 4><<<g2, PRED_THREADS, 0, st>>>(rows, F, Fpad, fr, dkf, cl, uvw, l, m, nm1,
                                                                                  flux, coh, station_form ? flag : nullptr);
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

extern "C" int sagecal_predict_set_form(int form) {
    if (form != 0 && form != 1) return SAGECAL_EINVAL;
    g_predict_form = form;
    return SAGECAL_OK;
}

extern "C" size_t sagecal_predict_workspace_bytes_station(int nstations, int ntime, int nchan, int nclus, int nsrc_total) {
    const size_t base = sagecal_predict_workspace_bytes(nchan, nsrc_total);
    if (base == 0 || nstations < 2 || ntime < 1 || nclus < 0) return base;
    const int ft = pick_ft(nchan);
    const int Fpad = (int)round_up((size_t)nchan, ft);
    const int npairs = nsrc_total / 2 + nclus;         // an upper bound: every cluster may end in a padding source
    const size_t per_slot = pg_bytes_per_slot(nstations, npairs, Fpad);
    const size_t cap = (size_t)2 << 30;                // the time slots are predicted in chunks of what fits 2 GiB
    size_t extra = per_slot * (size_t)ntime;
    if (extra > cap) extra = per_slot * (cap / per_slot > 0 ? cap / per_slot : 1);
    return base + round_up(extra, 256);
}

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
    // the last 256 bytes of the workspace: the device-side flag "uvw are not station differences"
    int* flag = (int*)((char*)flux + round_up(sizeof(double) * (size_t)S * Fpad * 4, 256));
    // whatever the caller gave beyond sagecal_predict_workspace_bytes(): room for the station phasors (station form)
    const size_t base_bytes = sagecal_predict_workspace_bytes(F, S);
    void* extra = workspace_bytes > base_bytes ? (void*)((char*)workspace + base_bytes) : nullptr;
    const size_t extra_bytes = extra ? workspace_bytes - base_bytes : 0;
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
                                                                    src_m, nm1, flux, coh, rs, N, T, flag, extra, extra_bytes); \
        return launch_predict<FT_, POL_, UNI_, SC_, false>(grid, st, rows, F, Fpad, fr, dkf, cl, uvw, src_l, src_m,    \
                                                          nm1, flux, coh, rs, N, T, flag, extra, extra_bytes);        \
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
                        src_alpha, coh_format, coh, precision, scratch, need, stream, nullptr);   // `need`: no room for station phasors -> per baseline
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
